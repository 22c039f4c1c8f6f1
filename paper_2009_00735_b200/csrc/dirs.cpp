// dirs.cpp -- step a3, host side: direction grids in fp64, stored as fp32 (include/aptsig.h).
// Fibonacci sphere: BASELINE.json configs 1-2 (not in the paper).  Geodesic sphere: the paper's
// "geodesic sphere finite element mesh" with N_v = 40 962 nodes = level 6.
#include <cmath>
#include <array>
#include <cstdint>
#include <cstring>
#include <map>
#include <unordered_map>
#include <vector>
#include "../../include/aptsig.h"

extern "C" int apx_dirs_fibonacci(int32_t D, float *out)
{
    if (D < 1 || !out) return APX_EINVAL;
    const double golden_angle = M_PI * (3.0 - std::sqrt(5.0));
    for (int32_t i = 0; i < D; ++i) {
        double z = 1.0 - (2.0 * (double)i + 1.0) / (double)D;
        double r = std::sqrt(std::fmax(0.0, 1.0 - z * z));
        double phi = (double)i * golden_angle;
        out[3 * (size_t)i + 0] = (float)(r * std::cos(phi));
        out[3 * (size_t)i + 1] = (float)(r * std::sin(phi));
        out[3 * (size_t)i + 2] = (float)z;
    }
    return APX_OK;
}

namespace {
struct V3 { double x, y, z; };
struct Tri { int a, b, c; };
}

extern "C" int apx_dirs_geodesic(int32_t level, float *out, int32_t *D_out)
{
    if (level < 0 || level > 8) return APX_EINVAL;
    int64_t nv = 2;
    { int64_t f = 10; for (int l = 0; l < level; ++l) f *= 4; nv += f; }
    if (D_out) *D_out = (int32_t)nv;
    if (!out) return D_out ? APX_OK : APX_EINVAL;

    const double t = (1.0 + std::sqrt(5.0)) / 2.0, inv = 1.0 / std::sqrt(1.0 + t * t);
    std::vector<V3> v = {{-1, t, 0}, {1, t, 0}, {-1, -t, 0}, {1, -t, 0}, {0, -1, t}, {0, 1, t},
                         {0, -1, -t}, {0, 1, -t}, {t, 0, -1}, {t, 0, 1}, {-t, 0, -1}, {-t, 0, 1}};
    for (auto &p : v) { p.x *= inv; p.y *= inv; p.z *= inv; }
    std::vector<Tri> f = {{0, 11, 5}, {0, 5, 1}, {0, 1, 7}, {0, 7, 10}, {0, 10, 11}, {1, 5, 9}, {5, 11, 4},
                          {11, 10, 2}, {10, 7, 6}, {7, 1, 8}, {3, 9, 4}, {3, 4, 2}, {3, 2, 6}, {3, 6, 8},
                          {3, 8, 9}, {4, 9, 5}, {2, 4, 11}, {6, 2, 10}, {8, 6, 7}, {9, 8, 1}};
    v.reserve((size_t)nv);
    for (int l = 0; l < level; ++l) {
        std::unordered_map<uint64_t, int> cache;
        cache.reserve(f.size() * 2);
        auto mid = [&](int a, int b) {
            uint64_t key = a < b ? ((uint64_t)a << 32) | (uint32_t)b : ((uint64_t)b << 32) | (uint32_t)a;
            auto it = cache.find(key);
            if (it != cache.end()) return it->second;
            V3 m = {v[a].x + v[b].x, v[a].y + v[b].y, v[a].z + v[b].z};
            double n = std::sqrt(m.x * m.x + m.y * m.y + m.z * m.z);
            m.x /= n; m.y /= n; m.z /= n;
            v.push_back(m);
            int id = (int)v.size() - 1;
            cache.emplace(key, id);
            return id;
        };
        std::vector<Tri> nf;
        nf.reserve(f.size() * 4);
        for (const Tri &tr : f) {
            int ab = mid(tr.a, tr.b), bc = mid(tr.b, tr.c), ca = mid(tr.c, tr.a);
            nf.push_back({tr.a, ab, ca});
            nf.push_back({tr.b, bc, ab});
            nf.push_back({tr.c, ca, bc});
            nf.push_back({ab, bc, ca});
        }
        f.swap(nf);
    }
    if ((int64_t)v.size() != nv) return APX_EINVAL;
    for (size_t i = 0; i < v.size(); ++i) {
        out[3 * i + 0] = (float)v[i].x;
        out[3 * i + 1] = (float)v[i].y;
        out[3 * i + 2] = (float)v[i].z;
    }
    return APX_OK;
}

extern "C" int apx_dirs_antipodes(const float *dirs, int32_t D, int32_t *partner)
{
    if (!dirs || D < 1) return APX_EINVAL;
    auto key = [&](int32_t i, float sgn) {
        std::array<uint32_t, 3> k;
        for (int a = 0; a < 3; ++a) {
            float v = sgn * dirs[3 * (size_t)i + a];
            if (v == 0.0f) v = 0.0f;                             // -0 and +0 are the same component
            std::memcpy(&k[a], &v, 4);
        }
        return k;
    };
    std::map<std::array<uint32_t, 3>, int32_t> index;
    bool sym = true;
    for (int32_t i = 0; i < D; ++i)
        if (!index.emplace(key(i, 1.0f), i).second) sym = false;  // duplicate direction
    for (int32_t i = 0; i < D; ++i) {
        auto it = index.find(key(i, -1.0f));
        const int32_t j = (it == index.end() || it->second == i) ? -1 : it->second;
        if (j < 0) sym = false;
        if (partner) partner[i] = j;
    }
    return sym ? 1 : 0;
}
