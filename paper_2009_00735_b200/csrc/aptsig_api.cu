// aptsig_api.cu -- the C ABI declared in include/aptsig.h: plan object (step a0), argument checks,
// error mapping, host staging for apx_run_host.  No arithmetic of the method lives here except the
// derived constants of the plan (R2, s, scaled directions, twiddles).
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>
#include "common.cuh"

using namespace apx;


#define CU(p, call)                                   \
    do {                                              \
        cudaError_t e__ = (call);                     \
        if (e__ != cudaSuccess) {                     \
            (p)->last_cuda = (int)e__;                \
            return e__ == cudaErrorMemoryAllocation ? APX_ENOMEM : APX_ECUDA; \
        }                                             \
    } while (0)

// Entry points run on the plan's device and leave the caller's current device as they found it.
struct DeviceGuard {
    int prev = -1;
    cudaError_t err;
    explicit DeviceGuard(int dev)
    {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
    }
    ~DeviceGuard()
    {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};
#define ON_DEVICE(p) DeviceGuard guard__((p)->device); CU(p, guard__.err)

static int ensure_capacity(apx_plan *p, int64_t N)
{
    if (N <= p->capacity) return APX_OK;
    if (p->d_sorted) cudaFree(p->d_sorted);
    p->d_sorted = nullptr; p->capacity = 0;
    int64_t cap = N + N / 8 + 1024;
    CU(p, cudaMalloc(&p->d_sorted, (size_t)cap * sizeof(float4)));
    p->capacity = cap;
    return APX_OK;
}

static int grow(apx_plan *p, void **buf, int64_t *cap, int64_t bytes)
{
    if (bytes <= *cap) return APX_OK;
    if (*buf) cudaFree(*buf);
    *buf = nullptr; *cap = 0;
    CU(p, cudaMalloc(buf, (size_t)bytes));
    *cap = bytes;
    return APX_OK;
}

extern "C" int apx_plan_destroy(apx_plan *p)
{
    if (!p) return APX_OK;
    DeviceGuard guard(p->device);
    void *bufs[] = {p->dbg_centre, p->dbg_sig, p->d_refine_off, p->d_kaxis, p->d_fsp_list, p->d_dirs_scaled, p->d_twiddle, p->d_mma_table, p->d_mma_zero, p->d_mma_phase, p->d_dirs_sorted, p->d_dir_perm, p->d_dir_perm_mirror, p->d_fft_half, p->d_fft_partner, p->d_type_mask, p->d_grid, p->d_cell_start,
                    p->d_cell_cursor, p->d_scan_tiles, p->d_sorted, p->d_deferred, p->h2d_xyz, p->h2d_types, p->h2d_centres,
                    p->d2h_sig, p->d2h_counts};
    for (void *b : bufs)
        if (b) cudaFree(b);
    if (p->own_stream) cudaStreamDestroy(p->own_stream);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    for (int i = 0; i < 2; ++i) {
        if (p->slab_done[i]) cudaEventDestroy(p->slab_done[i]);
        if (p->copy_done[i]) cudaEventDestroy(p->copy_done[i]);
    }
    delete p;
    return APX_OK;
}

static int create_plan(const apx_plan_desc *desc, const apx_sig_spec *specs_in, int n_specs, apx_plan **out)
{
    if (!out) return APX_EINVAL;
    *out = nullptr;
    if (!desc || !desc->dirs || !specs_in || n_specs < 1 || n_specs > APX_MAX_SIGNATURES) return APX_EINVAL;
    const int B = desc->B;
    if (!(desc->R > 0.0f) || !std::isfinite(desc->R)) return APX_EINVAL;
    if (B < 256 || B > 4096 || (B & (B - 1))) return APX_EINVAL;
    if (desc->pad != 0 && desc->pad != 1) return APX_EINVAL;
    if (desc->D < 1) return APX_EINVAL;
    if ((desc->flags & APX_FLAG_FORCE_FFT) && (desc->flags & APX_FLAG_FORCE_MMA)) return APX_EINVAL;
    // specs -> classes (distinct type masks), union window, union type mask
    SpecSet ss;
    std::memset(&ss, 0, sizeof(ss));
    ss.n_specs = n_specs;
    int k_lo = B, k_hi = -1;
    bool any_local = false;
    uint32_t union_mask[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = 0; i < n_specs; ++i) {
        int lo = specs_in[i].k_lo, hi = specs_in[i].k_hi;
        if (lo == 0 && hi == 0) { lo = 1; hi = B / 2; }
        if (lo < 0 || hi > B / 2 || lo > hi) return APX_EINVAL;
        if (specs_in[i].peak_mode != APX_PEAK_MAX && specs_in[i].peak_mode != APX_PEAK_LOCAL_MAX) return APX_EINVAL;
        ss.k_lo[i] = lo; ss.k_hi[i] = hi; ss.mode[i] = specs_in[i].peak_mode; ss.norm[i] = specs_in[i].normalise ? 1 : 0;
        any_local = any_local || specs_in[i].peak_mode == APX_PEAK_LOCAL_MAX;
        k_lo = lo < k_lo ? lo : k_lo; k_hi = hi > k_hi ? hi : k_hi;
        uint32_t m[8];
        std::memcpy(m, specs_in[i].type_mask, 32);
        int cls = -1;
        for (int c = 0; c < ss.n_classes; ++c)
            if (!std::memcmp(ss.cls_mask[c], m, 32)) cls = c;
        if (cls < 0) { cls = ss.n_classes++; std::memcpy(ss.cls_mask[cls], m, 32); }
        ss.cls_of[i] = cls;
        for (int wd = 0; wd < 8; ++wd) union_mask[wd] |= m[wd];
    }
    if (any_local && (desc->flags & APX_FLAG_FORCE_MMA)) return APX_EINVAL;       // local-maximum mode: general kernel only

    apx_plan *p = new (std::nothrow) apx_plan();
    if (!p) return APX_ENOMEM;
    std::memset(static_cast<apx::Plan *>(p), 0, sizeof(apx::Plan));
    p->desc = *desc;
    p->desc.dirs = nullptr;
    p->B = B; p->D = desc->D; p->pad = desc->pad; p->k_lo = k_lo; p->k_hi = k_hi; p->W = k_hi - k_lo + 1;
    p->specs = ss;
    p->R = desc->R; p->device = desc->device;
    volatile float r2 = desc->R * desc->R;                                     // one fp32 multiply
    p->R2 = r2;
    p->s = (float)((double)(B / 2 - desc->pad) / (double)desc->R);             // fp64, rounded once

    auto fail = [&](int code) { apx_plan_destroy(p); return code; };
    DeviceGuard guard(p->device);
    if (guard.err != cudaSuccess) { delete p; return APX_ECUDA; }
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, p->device) != cudaSuccess) { delete p; return APX_ECUDA; }
    p->sm_count = prop.multiProcessorCount;

    // scaled directions n' = fl32(n * s), one fp32 multiply per component
    std::vector<float> nps((size_t)3 * p->D);
    for (size_t i = 0; i < nps.size(); ++i) { volatile float v = desc->dirs[i] * p->s; nps[i] = v; }
    std::vector<float2> tw((size_t)B / 2);
    for (int r = 0; r < B / 2; ++r) {
        double th = 2.0 * M_PI * (double)r / (double)B;
        tw[r] = make_float2((float)std::cos(th), (float)-std::sin(th));
    }
    uint32_t mask[8];
    std::memcpy(mask, union_mask, 32);                                         // ingest keeps every ion some spec accepts

#define CUF(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { p->last_cuda = (int)e__; \
        return fail(e__ == cudaErrorMemoryAllocation ? APX_ENOMEM : APX_ECUDA); } } while (0)
    CUF(cudaMalloc(&p->d_dirs_scaled, nps.size() * sizeof(float)));
    CUF(cudaMalloc(&p->d_twiddle, tw.size() * sizeof(float2)));
    CUF(cudaMalloc(&p->d_type_mask, 32));
    CUF(cudaMalloc(&p->d_grid, sizeof(GridParams)));
    CUF(cudaMalloc(&p->d_cell_start, (size_t)(kMaxCells + 1) * sizeof(uint32_t)));
    CUF(cudaMalloc(&p->d_cell_cursor, (size_t)kMaxCells * sizeof(uint32_t)));
    CUF(cudaMalloc(&p->d_scan_tiles, (size_t)(kMaxCells / 8192) * sizeof(uint32_t)));
    CUF(cudaMemcpy(p->d_dirs_scaled, nps.data(), nps.size() * sizeof(float), cudaMemcpyHostToDevice));
    CUF(cudaMemcpy(p->d_twiddle, tw.data(), tw.size() * sizeof(float2), cudaMemcpyHostToDevice));
    CUF(cudaMemcpy(p->d_type_mask, mask, 32, cudaMemcpyHostToDevice));
    CUF(cudaStreamCreateWithFlags(&p->own_stream, cudaStreamNonBlocking));
    CUF(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
    CUF(cudaEventCreateWithFlags(&p->slab_done[0], cudaEventDisableTiming));
    CUF(cudaEventCreateWithFlags(&p->slab_done[1], cudaEventDisableTiming));
    CUF(cudaEventCreateWithFlags(&p->copy_done[0], cudaEventDisableTiming));
    CUF(cudaEventCreateWithFlags(&p->copy_done[1], cudaEventDisableTiming));
    CUF(cudaMalloc(&p->dbg_centre, 16));

    // the clamp of Eq. 1's bin index can be skipped when it provably never triggers: paper padding (pad = 1) and
    // directions that are unit vectors to fp32 accuracy => |x| <= (B/2-1)(1+2e-5) < B/2 - 0.25
    {
        bool unit = p->pad == 1;
        const double lim = (double)p->s * 1.00001;
        for (int d = 0; d < p->D && unit; ++d) {
            const double nn = std::sqrt((double)nps[3 * d] * nps[3 * d] + (double)nps[3 * d + 1] * nps[3 * d + 1] +
                                        (double)nps[3 * d + 2] * nps[3 * d + 2]);
            if (!(nn <= lim)) unit = false;
        }
        p->need_clamp = unit ? 0 : 1;
    }
    // Half-grid mode of the general kernel (antipodally symmetric grids, e.g. the paper's geodesic mesh, L60): it bins the
    // lower-numbered member of every pair (n, -n) and writes the peak to both (signature_fft.cu).  Used whenever that kernel
    // runs: plans on the FFT path and the material points the tensor-core kernel defers.
    {
        const int D = p->D;
        std::vector<int32_t> partner((size_t)D, -1);
        if (!p->need_clamp && !(desc->flags & APX_FLAG_NO_PAIRING) && D >= 2 && D % 2 == 0 &&
            apx_dirs_antipodes(nps.data(), D, partner.data()) == 1) {
            std::vector<int32_t> half;
            half.reserve((size_t)D / 2);
            for (int d = 0; d < D; ++d)
                if (d < partner[d]) half.push_back(d);
            if ((int)half.size() == D / 2) {
                CUF(cudaMalloc(&p->d_fft_half, half.size() * 4));
                CUF(cudaMalloc(&p->d_fft_partner, partner.size() * 4));
                CUF(cudaMemcpy(p->d_fft_half, half.data(), half.size() * 4, cudaMemcpyHostToDevice));
                CUF(cudaMemcpy(p->d_fft_partner, partner.data(), partner.size() * 4, cudaMemcpyHostToDevice));
                p->fft_paired = 1;
            }
        }
    }
    p->path = 0;
    if (!(desc->flags & APX_FLAG_FORCE_FFT) && !any_local && mma_path_supported(p)) {
        CUF(mma_path_prepare(p));
        p->path = 1;
    } else if (desc->flags & APX_FLAG_FORCE_MMA) {
        return fail(APX_EINVAL);
    }
#undef CUF
    *out = p;
    return APX_OK;
}

extern "C" int apx_plan_create(const apx_plan_desc *desc, apx_plan **out)
{
    if (!out) return APX_EINVAL;
    *out = nullptr;
    if (!desc) return APX_EINVAL;
    apx_sig_spec one;
    std::memcpy(one.type_mask, desc->type_mask, 32);
    one.k_lo = desc->k_lo; one.k_hi = desc->k_hi;
    one.peak_mode = (desc->flags & APX_FLAG_LOCAL_MAX) ? APX_PEAK_LOCAL_MAX : APX_PEAK_MAX;
    one.normalise = (desc->flags & APX_FLAG_NORMALISE) ? 1 : 0;
    return create_plan(desc, &one, 1, out);
}

extern "C" int apx_plan_create_multi(const apx_plan_desc *desc, const apx_sig_spec *specs, int32_t n_specs, apx_plan **out)
{
    return create_plan(desc, specs, n_specs, out);
}

extern "C" int apx_plan_num_signatures(const apx_plan *p) { return p ? p->specs.n_specs : APX_EINVAL; }

extern "C" int apx_plan_constants(const apx_plan *p, float *R2, float *s, float *freq_per_bin)
{
    if (!p) return APX_EINVAL;
    if (R2) *R2 = p->R2;
    if (s) *s = p->s;
    if (freq_per_bin) *freq_per_bin = p->s / (float)p->B;
    return APX_OK;
}

extern "C" int apx_plan_path(const apx_plan *p) { return p ? p->path : APX_EINVAL; }
extern "C" int apx_plan_paired(const apx_plan *p) { return p ? (p->path == 1 ? p->mma_paired : p->fft_paired) : APX_EINVAL; }
extern "C" int apx_last_cuda_error(const apx_plan *p) { return p ? p->last_cuda : (int)cudaErrorInvalidValue; }

extern "C" int apx_ingest(apx_plan *p, const float *xyz, const uint8_t *types, int64_t N, void *stream)
{
    if (!p || N < 0 || (N > 0 && !xyz)) return APX_EINVAL;
    if (N >= (1LL << 31)) return APX_ERANGE;
    ON_DEVICE(p);
    int rc = ensure_capacity(p, N);
    if (rc) return rc;
    CU(p, launch_ingest(p, xyz, types, N, (cudaStream_t)stream));
    p->ingested = true;
    return APX_OK;
}

extern "C" int apx_query(apx_plan *p, const float *centres, int64_t M, float *sig, uint32_t *counts, void *stream)
{
    if (!p || M < 0 || (M > 0 && (!centres || !sig))) return APX_EINVAL;
    if (!p->ingested) return APX_ESTATE;
    if ((double)M * (double)p->D >= 1099511627776.0) return APX_ERANGE;
    ON_DEVICE(p);
    if (p->path == 1) CU(p, launch_signature_mma(p, centres, M, sig, counts, (cudaStream_t)stream));
    else CU(p, launch_signature_fft(p, centres, M, sig, counts, (cudaStream_t)stream));
    return APX_OK;
}

extern "C" int apx_run(apx_plan *p, const float *xyz, const uint8_t *types, int64_t N, const float *centres,
                       int64_t M, float *sig, uint32_t *counts, void *stream)
{
    int rc = apx_ingest(p, xyz, types, N, stream);
    if (rc) return rc;
    return apx_query(p, centres, M, sig, counts, stream);
}

extern "C" int apx_plan_reserve(apx_plan *p, int64_t N_max, int64_t M_max)
{
    if (!p || N_max < 0 || M_max < 0) return APX_EINVAL;
    if (N_max >= (1LL << 31)) return APX_ERANGE;
    ON_DEVICE(p);
    int rc = ensure_capacity(p, N_max);
    if (rc) return rc;
    if (p->path == 1) CU(p, mma_reserve_for(p, M_max));
    return APX_OK;
}

// Output staging of apx_run_host: two device slabs of at most kSlabBytes each, used alternately (slab i in buffer
// i & 1): the signatures of slab i travel to the host on the copy stream while slab i + 1 is computed.
static const int64_t kSlabBytes = 1LL << 30;

extern "C" int apx_run_host(apx_plan *p, const float *xyz, const uint8_t *types, int64_t N, const float *centres,
                            int64_t M, float *sig, uint32_t *counts)
{
    if (!p || N < 0 || M < 0 || (N > 0 && !xyz) || (M > 0 && (!centres || !sig))) return APX_EINVAL;
    if (N >= (1LL << 31)) return APX_ERANGE;
    ON_DEVICE(p);
    cudaStream_t st = p->own_stream;
    const int S = p->specs.n_specs;
    const int64_t row_bytes = (int64_t)p->D * 8 * S;              // all signature planes of one material point
    // material points per slab: bounded by the staging size, and at most a quarter of the job so that copies overlap
    int64_t slab = kSlabBytes / row_bytes;
    if (slab < 1) slab = 1;
    if (M > 128 && slab > (M + 3) / 4) slab = (M + 3) / 4;
    if (slab > M) slab = M > 0 ? M : 1;
    const int64_t nslab = M > 0 ? (M + slab - 1) / slab : 0;
    int rc;
    if ((rc = grow(p, &p->h2d_xyz, &p->cap_xyz, N * 12 + 16))) return rc;
    if (types && (rc = grow(p, &p->h2d_types, &p->cap_types, N + 16))) return rc;
    if ((rc = grow(p, &p->h2d_centres, &p->cap_centres, M * 12 + 16))) return rc;
    if ((rc = grow(p, &p->d2h_sig, &p->cap_sig, (nslab > 1 ? 2 : 1) * slab * row_bytes + 16))) return rc;
    if (counts && (rc = grow(p, &p->d2h_counts, &p->cap_counts, (nslab > 1 ? 2 : 1) * slab * 4 * S + 16))) return rc;
    if ((rc = ensure_capacity(p, N))) return rc;
    if (p->path == 1) CU(p, mma_reserve_for(p, slab));
    // from here on work is in flight on the two internal streams: never return before both have drained, the copies
    // read and write the caller's host buffers
    auto drain = [&](int code) {
        cudaStreamSynchronize(p->copy_stream);
        cudaStreamSynchronize(st);
        return code;
    };
#define CUD(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { p->last_cuda = (int)e__; \
        return drain(e__ == cudaErrorMemoryAllocation ? APX_ENOMEM : APX_ECUDA); } } while (0)
    if (N) CUD(cudaMemcpyAsync(p->h2d_xyz, xyz, (size_t)N * 12, cudaMemcpyHostToDevice, st));
    if (N && types) CUD(cudaMemcpyAsync(p->h2d_types, types, (size_t)N, cudaMemcpyHostToDevice, st));
    if (M) CUD(cudaMemcpyAsync(p->h2d_centres, centres, (size_t)M * 12, cudaMemcpyHostToDevice, st));
    rc = apx_ingest(p, (const float *)p->h2d_xyz, types ? (const uint8_t *)p->h2d_types : nullptr, N, st);
    if (rc) return drain(rc);
    for (int64_t m0 = 0, i = 0; m0 < M; m0 += slab, ++i) {
        const int64_t mc = (M - m0 < slab) ? M - m0 : slab;
        // a slab's staging holds its planes back to back: [S][mc][D][2] and [S][mc]
        float *dsig = (float *)p->d2h_sig + (i & 1) * slab * (int64_t)p->D * 2 * S;
        uint32_t *dcnt = counts ? (uint32_t *)p->d2h_counts + (i & 1) * slab * S : nullptr;
        if (i >= 2) CUD(cudaStreamWaitEvent(st, p->copy_done[i & 1], 0));       // the buffer's previous slab has left
        rc = apx_query(p, (const float *)p->h2d_centres + 3 * m0, mc, dsig, dcnt, st);
        if (rc) return drain(rc);
        CUD(cudaEventRecord(p->slab_done[i & 1], st));
        CUD(cudaStreamWaitEvent(p->copy_stream, p->slab_done[i & 1], 0));
        for (int sp = 0; sp < S; ++sp) {                              // plane sp of the slab -> plane sp of the caller's array
            CUD(cudaMemcpyAsync(sig + ((int64_t)sp * M + m0) * p->D * 2, dsig + (int64_t)sp * mc * p->D * 2,
                                (size_t)(mc * (int64_t)p->D * 8), cudaMemcpyDeviceToHost, p->copy_stream));
            if (counts) CUD(cudaMemcpyAsync(counts + (int64_t)sp * M + m0, dcnt + (int64_t)sp * mc, (size_t)mc * 4,
                                            cudaMemcpyDeviceToHost, p->copy_stream));
        }
        CUD(cudaEventRecord(p->copy_done[i & 1], p->copy_stream));
    }
#undef CUD
    CU(p, cudaStreamSynchronize(p->copy_stream));
    CU(p, cudaStreamSynchronize(st));
    return APX_OK;
}

// Test hook: ONE material point through the plan's production kernel (the one apx_query launches: tensor-core or FFT
// path, half-grid mode, spill / multi-pass / deferred handling included) with the histogram export switched on.
extern "C" int apx_debug_histograms(apx_plan *p, const float *centre3, int32_t d0, int32_t nd, uint32_t *out,
                                    void *stream)
{
    if (!p || !centre3 || d0 < 0 || nd < 0 || d0 + nd > p->D || (nd > 0 && !out)) return APX_EINVAL;
    if (!p->ingested) return APX_ESTATE;
    if (nd == 0) return APX_OK;
    ON_DEVICE(p);
    cudaStream_t st = (cudaStream_t)stream;
    int rc;
    int64_t cap = p->dbg_sig ? (int64_t)p->D * 8 * p->specs.n_specs : 0;
    if ((rc = grow(p, (void **)&p->dbg_sig, &cap, (int64_t)p->D * 8 * p->specs.n_specs))) return rc;
    CU(p, cudaMemcpyAsync(p->dbg_centre, centre3, 12, cudaMemcpyHostToDevice, st));
    CU(p, cudaMemsetAsync(out, 0, (size_t)nd * p->B * sizeof(uint32_t), st));
    p->dbg_hist_out = out; p->dbg_d0 = d0; p->dbg_nd = nd;
    rc = apx_query(p, p->dbg_centre, 1, p->dbg_sig, nullptr, st);
    p->dbg_hist_out = nullptr; p->dbg_d0 = 0; p->dbg_nd = 0;
    return rc;
}

#ifdef APX_TRACE
// development builds only: the tensor-core path's slot order (original direction index per slot, -1 = padding)
extern "C" int apx_debug_slot_order(apx_plan *p, int *perm, int *mirror)
{
    if (!p || p->path != 1) return APX_EINVAL;
    if (perm) cudaMemcpy(perm, p->d_dir_perm, (size_t)p->Dp * 4, cudaMemcpyDeviceToHost);
    if (mirror && p->d_dir_perm_mirror) cudaMemcpy(mirror, p->d_dir_perm_mirror, (size_t)p->Dp * 4, cudaMemcpyDeviceToHost);
    return p->Dp;
}
// development builds only (-DAPX_TRACE, not declared in the public headers): timeline buffer for k_signature_mma
extern "C" int apx_debug_trace(apx_plan *p, long long *device_buf, int block, int cap)
{
    if (!p) return APX_EINVAL;
    p->dbg_trace = device_buf; p->dbg_trace_block = block; p->dbg_trace_cap = cap;
    return APX_OK;
}
#endif

extern "C" const char *apx_strerror(int s)
{
    switch (s) {
        case APX_OK: return "ok";
        case APX_EINVAL: return "invalid argument";
        case APX_ENOMEM: return "out of memory";
        case APX_ECUDA: return "CUDA error (see apx_last_cuda_error)";
        case APX_ESTATE: return "no ion cloud ingested";
        case APX_ERANGE: return "size out of range";
        default: return "unknown status";
    }
}

extern "C" const char *apx_version(void) { return "aptsig 0.1 (sm_100a)"; }
