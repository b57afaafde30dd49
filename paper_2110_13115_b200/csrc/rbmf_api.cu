// The C ABI of librbmf.so (include/rbmf.h): plan management, workspace layout, TMA descriptors, launch sequence.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "rbmf_internal.h"

using namespace rbmf;

namespace {

constexpr size_t kAlign = 1024;
inline size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }
inline int ilog2(int64_t x) { int l = 0; while ((int64_t(1) << l) < x) ++l; return l; }

// One instance of kernel 1 working on `ncols` columns of length-N series (the template routes run two besides the
// plan's own: full length for the flat method, length 2 N / w for the fast first stage).
struct TmUnit {
    int64_t N;
    int logN1, logN2, ncols;
    size_t basisP, beta, tw1_a, tw1_b, twN, dsT, sched;   // workspace offsets
    CUtensorMap tmY;
};

struct Layout {
    size_t basisP, beta, bavg_hi, bavg_lo, c_hi, c_lo, c_h16, tnorm_blk, bin_norm, cs, tw1_a, tw1_b, twN, dsT,
        cand, cand2, cand3, bin_count, bin_start, items, counters, sched, strain_stage, trig_stage, twF, r2c_s, r2c_z, tm_S, tm_isg, total;
    size_t sched_bytes;
    size_t plane_bytes;
};

}  // namespace

struct rbmf_plan {
    int64_t N;
    double fs, f_low;
    int k, T, w;
    int64_t M;          // N / w
    int j_low, n_half;
    int Tpad;
    int logN1, logN2;   // FFT: N = 2^logN1 * 2^logN2 (pass 1 length, pass 2 length)
    int fft_grid;       // persistent CTAs of the fused FFT kernel
    int64_t max_cand, max_trig;
    int max_batch;      // segments rbmf_filter_batch may take at once (rbmf_plan_set_batch; default 1)
    int last_nb;        // segments of the last rbmf_filter / rbmf_filter_batch
    int gemm_impl;
    int last_impl;      // gemm_impl of the last rbmf_filter (decides which candidate list / counter is final)
    int diag_fp32_check, diag_single_cta, diag_stage2_per_cand;   // rbmf_diag_set
    int diag_fft_chunk_major, diag_fft_lookahead, diag_gemm_group;   // rbmf_diag_set: scheduling overrides, 0 = automatic
    int timing;
    cudaStream_t stream;
    uint8_t* ws;
    size_t ws_bytes;
    Layout lay;
    bool have_ws, have_basis, have_coeffs, filtered;
    int num_sms;
    int last_cuda;
    CUtensorMap tmA_hi, tmA_lo, tmB_hi, tmB_lo, tmB_h16, tmB_h16half, tmY;
    int pair_clusters;   // 2-CTA clusters of the screen GEMM the device holds (0: single-CTA kernel)
    // template routes (rbmf_plan_enable_template_routes): slab = templates per pass (0 = disabled)
    int tm_slab, stage1_route;
    TmUnit tmF, tmS;     // flat method: length N; fast first stage: length 2 N / w
    const void* tm_templates;   // caller's T x (N/2+1) bank (retained pointer)
    // bank sets (rbmf_bankset_*): a trigger list and position counter shared with other plans, sub-bank id offset
    unsigned long long* shared_trig_counter;
    unsigned long long shared_trig_cap;
    int template_offset;
    bool have_templates;
    bool have_maps;
    cudaEvent_t ev[kEvRing][4];   // stage events of the last kEvRing timed calls (ring; ev_slot = the latest)
    int ev_slot;
    long long ev_calls;           // timed calls since timing was switched on
    bool have_events;
};

namespace {

Layout make_layout(const rbmf_plan* p) {
    Layout L;
    size_t off = 0;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
    const size_t k = (size_t)p->k, N = (size_t)p->N, B = (size_t)p->max_batch;
    const size_t M = (size_t)p->M * B;   // rows of the planes: all segments of a batch, segment-major
    const size_t nkb = (k + 31) / 32;
    L.plane_bytes = nkb * M * 64 * 2;
    // pass-1 tile inputs in tile-buffer order (rbmf_internal.h): k L2 fft_p1_rows(L1) basis values, L2 strain rows
    L.basisP = take(k * ((size_t)1 << p->logN2) * (size_t)fft_p1_rows(p->logN1) * 8);
    L.beta = take(B * N * k * 8);
    L.bavg_hi = take(L.plane_bytes);
    L.bavg_lo = take(L.plane_bytes);
    L.c_hi = take((size_t)p->Tpad * 2 * 2 * k * 2);
    L.c_lo = take((size_t)p->Tpad * 2 * 2 * k * 2);
    L.c_h16 = take((size_t)p->Tpad * 2 * 2 * k * 2);
    L.tnorm_blk = take((size_t)(p->Tpad / kGemmTT) * 4);
    L.bin_norm = take(M * 4);
    L.cs = take((size_t)p->T * k * 8);
    L.tw1_a = take(((size_t)1 << p->logN1) * 8);
    L.tw1_b = take(((size_t)1 << p->logN2) * 8);
    L.twN = take(((size_t)1 << p->logN2) * (size_t)(fft_r0(p->logN1) + fft_r1(p->logN1)) * 8);   // two factor tables
    L.dsT = take(B * ((size_t)1 << p->logN2) * (size_t)fft_strain_row(p->logN1) * 8);
    L.cand = take((size_t)p->max_cand * sizeof(rbmf_candidate));
    L.cand2 = take((size_t)p->max_cand * sizeof(rbmf_candidate));
    L.cand3 = take((size_t)p->max_cand * sizeof(rbmf_candidate));
    L.bin_start = take(M * 4);
    L.items = take(((size_t)p->max_cand / kStage2Chunk + M + 1) * sizeof(int4));
    // counters, the FFT scheduler words and the per-bin histogram are contiguous: one memset per call
    L.sched_bytes = ((size_t)kSchedBase + (size_t)kMaxChunks * B) * 4;
    L.counters = take(kCounterBytes + L.sched_bytes + M * 4);
    L.sched = L.counters + kCounterBytes;
    L.bin_count = L.sched + L.sched_bytes;
    L.strain_stage = take(B * (size_t)(p->n_half + 1) * 8);
    L.trig_stage = take((size_t)p->max_trig * sizeof(rbmf_trigger));
    L.twF = take((size_t)p->n_half * 8);                 // front end: e^{-2 pi i m / N}, m < N/2
    L.r2c_s = take(B * (size_t)p->n_half * 8);
    L.r2c_z = take(B * (size_t)p->n_half * 8);
    if (p->tm_slab > 0) {
        L.tm_S = take((size_t)p->n_half * 8);
        L.tm_isg = take((size_t)p->T * 4);
        TmUnit* units[2] = {const_cast<TmUnit*>(&p->tmF), const_cast<TmUnit*>(&p->tmS)};
        for (int u = 0; u < 2; ++u) {
            TmUnit& U = *units[u];
            U.N = u == 0 ? p->N : 2 * p->N / p->w;
            const int n = ilog2(U.N);
            U.logN1 = (n + 1) / 2; U.logN2 = n / 2; U.ncols = p->tm_slab;
            U.basisP = take((size_t)U.ncols * ((size_t)1 << U.logN2) * (size_t)fft_p1_rows(U.logN1) * 8);
            U.beta = take((size_t)U.N * U.ncols * 8);
            U.tw1_a = take(((size_t)1 << U.logN1) * 8);
            U.tw1_b = take(((size_t)1 << U.logN2) * 8);
            U.twN = take(((size_t)1 << U.logN2) * (size_t)(fft_r0(U.logN1) + fft_r1(U.logN1)) * 8);
            U.dsT = take(((size_t)1 << U.logN2) * (size_t)fft_strain_row(U.logN1) * 8);
            U.sched = take(((size_t)kSchedBase + kMaxChunks) * 4);
        }
    }
    L.total = off;
    return L;
}

void refresh(rbmf_plan* p) {
    p->M = p->N / p->w;
    const int n = ilog2(p->N);
    p->logN1 = (n + 1) / 2; p->logN2 = n / 2;
    p->Tpad = (p->T + kGemmTT - 1) / kGemmTT * kGemmTT;
    p->lay = make_layout(p);
}

rbmf_status cuda_fail(rbmf_plan* p, cudaError_t e) {
    if (p) p->last_cuda = (int)e;
    return RBMF_ERR_CUDA;
}

#define CK(call)                                              \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(plan, e__);  \
    } while (0)

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

rbmf_status encode_map(rbmf_plan* plan, CUtensorMap* map, void* base, int rank, const cuuint64_t* dims,
                       const cuuint64_t* strides, const cuuint32_t* box,
                       CUtensorMapDataType dtype = CU_TENSOR_MAP_DATA_TYPE_BFLOAT16,
                       CUtensorMapSwizzle swizzle = CU_TENSOR_MAP_SWIZZLE_128B) {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres);
        if (e != cudaSuccess) return cuda_fail(plan, e);
        if (qres != cudaDriverEntryPointSuccess || !sym) { plan->last_cuda = -1; return RBMF_ERR_CUDA; }
        fn = (EncodeTiledFn)sym;
    }
    const cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(map, dtype, (cuuint32_t)rank, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { plan->last_cuda = (int)r; return RBMF_ERR_CUDA; }
    return RBMF_OK;
}

// Coefficient planes: rows x cols bf16, row-major; box = 64 columns x box_rows.
rbmf_status make_map_rows(rbmf_plan* plan, CUtensorMap* map, void* base, uint64_t rows, uint64_t cols,
                          uint32_t box_rows) {
    const cuuint64_t dims[2] = {cols, rows};               // innermost first
    const cuuint64_t strides[1] = {cols * 2};              // bytes, dims 1..rank-1
    const cuuint32_t box[2] = {(cuuint32_t)kGemmBK, box_rows};
    return encode_map(plan, map, base, 2, dims, strides, box);
}

// beta^avg planes: [kb][bin < M][64] bf16; box = one K block x 128 bins (16 KB contiguous).
rbmf_status make_map_planes(rbmf_plan* plan, CUtensorMap* map, void* base, uint64_t M, uint64_t nkb) {
    const cuuint64_t dims[3] = {(cuuint64_t)kGemmBK, M, nkb};
    const cuuint64_t strides[2] = {(cuuint64_t)kGemmBK * 2, M * kGemmBK * 2};
    const cuuint32_t box[3] = {(cuuint32_t)kGemmBK, (cuuint32_t)kGemmBM, 1};
    return encode_map(plan, map, base, 3, dims, strides, box);
}

// Y rows of a pass-2 FFT tile: the beta array viewed as fp32 [chunk][j2 < L2][2 C L1] (Y[n1][j2] sits at the address
// of beta[n1 + L1 j2]); box = sub2 lines x C columns (re, im) wide, up to 256 rows j2, unswizzled.
rbmf_status make_map_y(rbmf_plan* plan, CUtensorMap* map, void* base, int logN1, int logN2, uint64_t nblocks) {
    const uint64_t L1 = 1ull << logN1, L2 = 1ull << logN2;
    const cuuint64_t dims[3] = {2 * kFftC * L1, L2, (cuuint64_t)nblocks};
    const cuuint64_t strides[2] = {L1 * kFftC * 8, (cuuint64_t)(L1 * L2) * kFftC * 8};
    const cuuint32_t box[3] = {(cuuint32_t)(2 * kFftC * fft_sub(logN2)), (cuuint32_t)(L2 < 256 ? L2 : 256), 1};
    return encode_map(plan, map, base, 3, dims, strides, box, CU_TENSOR_MAP_DATA_TYPE_FLOAT32,
                      CU_TENSOR_MAP_SWIZZLE_NONE);
}

template <typename T> T* at(rbmf_plan* p, size_t off) { return reinterpret_cast<T*>(p->ws + off); }

}  // namespace

// ---- template routes ------------------------------------------------------------------------
namespace {

// One launch of kernel 1 on a template-route unit: ncols columns, one segment, no operand planes.
rbmf_status run_tm_unit(rbmf_plan* plan, const TmUnit& U) {
    cudaStream_t st = plan->stream;
    CK(cudaMemsetAsync(plan->ws + U.sched, 0, ((size_t)kSchedBase + kMaxChunks) * 4, st));
    FftArgs a;
    memset(&a, 0, sizeof(a));
    a.basisP = at<float2>(plan, U.basisP); a.dsT = at<float2>(plan, U.dsT);
    a.tw1_a = at<float2>(plan, U.tw1_a); a.tw1_b = at<float2>(plan, U.tw1_b); a.twN = at<float2>(plan, U.twN);
    a.beta = at<float2>(plan, U.beta);
    a.sched = at<unsigned>(plan, U.sched);
    a.N = U.N; a.M = (int)U.N; a.Mseg = (int)U.N; a.nb = 1; a.nchunk = U.ncols / kFftC; a.w = 1; a.inv_w = 1.f;
    a.no_planes = 1;
    const long long n1t = (1ll << U.logN2) / fft_sub(U.logN1);
    long long la = (4ll * plan->fft_grid + n1t - 1) / n1t;
    const long long cap = (48ll << 20) / ((long long)U.N * kFftC * 8) - 1;
    if (la > cap) la = cap;
    if (la < 1) la = 1;
    a.lookahead = (int)la;
    CK(launch_fft_tma(U.tmY, a, U.logN1, U.logN2, plan->fft_grid, st));
    return RBMF_OK;
}

// Fast first stage by templates (Eq. 10-12): fold -> short transform -> threshold scan, slab by slab; fills the
// stage-1 list, counters[0] and the per-bin histogram exactly like kernel 2 does.
rbmf_status stage1_by_templates(rbmf_plan* plan, const float2* strain_dev, float thr1) {
    const Layout& L = plan->lay;
    const TmUnit& U = plan->tmS;
    unsigned long long* counters = at<unsigned long long>(plan, L.counters);
    const float scale = (float)sqrt(2.0 / (double)plan->N);
    for (int t0 = 0; t0 < plan->T; t0 += U.ncols) {
        CK(launch_tm_fold((const float2*)plan->tm_templates, strain_dev, at<float2>(plan, L.tm_S),
                          at<float2>(plan, U.basisP), plan->N / 2 + 1, plan->j_low, plan->n_half, plan->w, scale, t0,
                          plan->T, U.ncols, U.logN1, U.logN2, fft_sub(U.logN1), plan->stream));
        rbmf_status s = run_tm_unit(plan, U);
        if (s != RBMF_OK) return s;
        CK(launch_tm_scan(at<float2>(plan, U.beta), U.N, 2, (int)plan->M, at<float>(plan, L.tm_isg), t0, plan->T,
                          U.ncols, thr1 * thr1, (rbmf_trigger*)at<rbmf_candidate>(plan, L.cand), counters,
                          (unsigned long long)plan->max_cand, at<unsigned>(plan, L.bin_count), plan->stream));
    }
    return RBMF_OK;
}

}  // namespace

extern "C" {

rbmf_status rbmf_plan_create(rbmf_plan** out, int64_t N, double fs, double f_low, int32_t k, int32_t T) {
    if (!out) return RBMF_ERR_ARG;
    *out = nullptr;
    if (N < 1024 || N > (int64_t(1) << 24) || (N & (N - 1)) != 0) return RBMF_ERR_ARG;
    if (!(fs > 0.0) || !(f_low > 0.0) || !(f_low < fs / 2)) return RBMF_ERR_ARG;
    if (k < 16 || k > 1024 || (k % 16) != 0) return RBMF_ERR_ARG;
    if (T < 1 || T > (1 << 24)) return RBMF_ERR_ARG;
    if (N > (int64_t(1) << 20)) return RBMF_ERR_UNSUPPORTED;   // valid, but the FFT is two passes of length <= 1024
    rbmf_plan* p = new (std::nothrow) rbmf_plan;
    if (!p) return RBMF_ERR_ARG;
    memset(p, 0, sizeof(*p));
    p->N = N; p->fs = fs; p->f_low = f_low; p->k = k; p->T = T;
    p->w = 8;
    p->n_half = (int)(N / 2);
    p->j_low = (int)ceil(f_low * (double)N / fs - 1e-12);
    if (p->j_low >= p->n_half) { delete p; return RBMF_ERR_ARG; }
    p->max_cand = int64_t(1) << 22;
    p->max_trig = int64_t(1) << 22;
    p->max_batch = 1;
    p->gemm_impl = RBMF_GEMM_SCREEN;
    refresh(p);
    *out = p;
    return RBMF_OK;
}

rbmf_status rbmf_plan_set_window(rbmf_plan* plan, int32_t w) {
    if (!plan) return RBMF_ERR_ARG;
    if (plan->have_ws) return RBMF_ERR_STATE;
    if (w < 1 || w > 32 || (w & (w - 1)) != 0) return RBMF_ERR_ARG;
    if (plan->N / w < kGemmBM) return RBMF_ERR_ARG;
    plan->w = w;
    refresh(plan);
    return RBMF_OK;
}

rbmf_status rbmf_plan_set_capacity(rbmf_plan* plan, int64_t max_candidates, int64_t max_triggers) {
    if (!plan) return RBMF_ERR_ARG;
    if (plan->have_ws) return RBMF_ERR_STATE;
    if (max_candidates < 1 || max_triggers < 1 || max_candidates > (int64_t(1) << 31) ||
        max_triggers > (int64_t(1) << 31))
        return RBMF_ERR_ARG;
    plan->max_cand = max_candidates;
    plan->max_trig = max_triggers;
    refresh(plan);
    return RBMF_OK;
}

rbmf_status rbmf_plan_set_batch(rbmf_plan* plan, int32_t max_batch) {
    if (!plan) return RBMF_ERR_ARG;
    if (plan->have_ws) return RBMF_ERR_STATE;
    // time_index = segment * N + n is an int32
    if (max_batch < 1 || (int64_t)max_batch * plan->N > (int64_t(1) << 31) - 1) return RBMF_ERR_ARG;
    plan->max_batch = max_batch;
    refresh(plan);
    return RBMF_OK;
}

rbmf_status rbmf_plan_set_gemm_impl(rbmf_plan* plan, int32_t impl) {
    if (!plan) return RBMF_ERR_ARG;
    if (impl != RBMF_GEMM_TCGEN05 && impl != RBMF_GEMM_SCREEN) return RBMF_ERR_ARG;
    plan->gemm_impl = impl;
    return RBMF_OK;
}

rbmf_status rbmf_workspace_bytes(const rbmf_plan* plan, size_t* bytes) {
    if (!plan || !bytes) return RBMF_ERR_ARG;
    *bytes = plan->lay.total;
    return RBMF_OK;
}

rbmf_status rbmf_set_stream(rbmf_plan* plan, void* cuda_stream) {
    if (!plan) return RBMF_ERR_ARG;
    plan->stream = (cudaStream_t)cuda_stream;
    return RBMF_OK;
}

rbmf_status rbmf_plan_set_workspace(rbmf_plan* plan, void* dev_ptr, size_t bytes) {
    if (!plan || !dev_ptr) return RBMF_ERR_ARG;
    if (((uintptr_t)dev_ptr % kAlign) != 0 || bytes < plan->lay.total) return RBMF_ERR_ARG;
    int dev = 0;
    CK(cudaGetDevice(&dev));
    int major = 0, minor = 0;
    CK(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    CK(cudaDeviceGetAttribute(&minor, cudaDevAttrComputeCapabilityMinor, dev));
    if (major != 10) return RBMF_ERR_UNSUPPORTED;   // sm_100a only: tcgen05 / TMEM
    CK(cudaDeviceGetAttribute(&plan->num_sms, cudaDevAttrMultiProcessorCount, dev));
    // the plan counts as ready only when every step below has succeeded
    plan->have_ws = plan->have_maps = false;
    plan->have_basis = plan->have_coeffs = plan->filtered = false;
    plan->ws = (uint8_t*)dev_ptr;
    plan->ws_bytes = bytes;
    const Layout& L = plan->lay;
    CK(launch_init_tables(at<float2>(plan, L.tw1_a), at<float2>(plan, L.tw1_b), at<float2>(plan, L.twN), plan->logN1,
                          plan->logN2, plan->stream));
    CK(cudaMemsetAsync(plan->ws + L.counters, 0, kCounterBytes + L.sched_bytes + (size_t)plan->M * plan->max_batch * 4,
                       plan->stream));
    // columns of the last K block beyond k are never written by the FFT: they must be finite (they meet zeros)
    CK(cudaMemsetAsync(plan->ws + L.bavg_hi, 0, L.plane_bytes, plan->stream));
    CK(cudaMemsetAsync(plan->ws + L.bavg_lo, 0, L.plane_bytes, plan->stream));
    CK(gemm_tcgen05_configure());
    CK(r2c_configure());
    CK(launch_r2c_table(at<float2>(plan, L.twF), plan->N, plan->stream));
    {
        size_t smem = 0;
        CK(fft_tma_configure(plan->logN1, plan->logN2, &smem));
        plan->fft_grid = plan->num_sms;   // persistent: one CTA (two consumer groups + a producer warp) per SM
    }
    // TMA descriptors: A = beta^avg planes ([kb][M][64]), B = coefficient planes (2*Tpad rows x 2k)
    rbmf_status s;
    const uint64_t k2 = 2 * (uint64_t)plan->k;
    const uint64_t nkb = (uint64_t)((plan->k + 31) / 32);
    if ((s = make_map_y(plan, &plan->tmY, plan->ws + L.beta, plan->logN1, plan->logN2,
                        (uint64_t)(plan->k / kFftC) * (uint64_t)plan->max_batch)) != RBMF_OK) return s;
    if (plan->tm_slab > 0) {
        TmUnit* units[2] = {&plan->tmF, &plan->tmS};
        for (int u = 0; u < 2; ++u) {
            TmUnit& U = *units[u];
            size_t smem = 0;
            CK(fft_tma_configure(U.logN1, U.logN2, &smem));
            CK(launch_init_tables(at<float2>(plan, U.tw1_a), at<float2>(plan, U.tw1_b), at<float2>(plan, U.twN),
                                  U.logN1, U.logN2, plan->stream));
            if ((s = make_map_y(plan, &U.tmY, plan->ws + U.beta, U.logN1, U.logN2, (uint64_t)(U.ncols / kFftC))) != RBMF_OK)
                return s;
        }
        // S(f) of Eq. 11; the fast first stage feeds its folded spectrum to kernel 1 with a unit "strain"
        CK(launch_tm_tables(at<float2>(plan, L.tm_S), at<float2>(plan, plan->tmS.dsT), plan->N, plan->w,
                            ((long long)1 << plan->tmS.logN2) * fft_strain_row(plan->tmS.logN1), plan->stream));
    }
    plan->have_templates = false;
    const uint64_t Mplane = (uint64_t)plan->M * (uint64_t)plan->max_batch;
    if ((s = make_map_planes(plan, &plan->tmA_hi, plan->ws + L.bavg_hi, Mplane, nkb)) != RBMF_OK) return s;
    if ((s = make_map_planes(plan, &plan->tmA_lo, plan->ws + L.bavg_lo, Mplane, nkb)) != RBMF_OK) return s;
    if ((s = make_map_rows(plan, &plan->tmB_hi, plan->ws + L.c_hi, 2 * (uint64_t)plan->Tpad, k2, 2 * kGemmTT)) != RBMF_OK) return s;
    if ((s = make_map_rows(plan, &plan->tmB_lo, plan->ws + L.c_lo, 2 * (uint64_t)plan->Tpad, k2, 2 * kGemmTT)) != RBMF_OK) return s;
    // fp16 data through a 16-bit tensor map: TMA only moves bytes, the element type is irrelevant without OOB fill
    if ((s = make_map_rows(plan, &plan->tmB_h16, plan->ws + L.c_h16, 2 * (uint64_t)plan->Tpad, k2, 2 * kGemmTT)) != RBMF_OK) return s;
    if ((s = make_map_rows(plan, &plan->tmB_h16half, plan->ws + L.c_h16, 2 * (uint64_t)plan->Tpad, k2, kGemmTT)) != RBMF_OK) return s;
    CK(gemm_screen_pair_clusters(plan->num_sms, &plan->pair_clusters));
    if (!plan->have_events) {
        for (int r = 0; r < kEvRing; ++r)
            for (int i = 0; i < 4; ++i) CK(cudaEventCreate(&plan->ev[r][i]));
        plan->have_events = true;
    }
    plan->have_maps = true;
    plan->have_ws = true;
    return RBMF_OK;
}

rbmf_status rbmf_set_basis(rbmf_plan* plan, const void* basis_dev) {
    if (!plan || !basis_dev) return RBMF_ERR_ARG;
    if (!plan->have_ws) return RBMF_ERR_STATE;
    CK(launch_layout_basis((const float2*)basis_dev, at<float2>(plan, plan->lay.basisP), plan->k, plan->N / 2 + 1,
                           plan->j_low, plan->logN1, plan->logN2, fft_sub(plan->logN1), plan->k, plan->stream));
    plan->have_basis = true;
    return RBMF_OK;
}

rbmf_status rbmf_set_coeffs(rbmf_plan* plan, const void* coeffs_dev, const float* sigma_dev) {
    if (!plan || !coeffs_dev) return RBMF_ERR_ARG;
    if (!plan->have_ws) return RBMF_ERR_STATE;
    const Layout& L = plan->lay;
    CK(launch_prep_coeffs((const float2*)coeffs_dev, sigma_dev, at<float2>(plan, L.cs), at<uint16_t>(plan, L.c_hi),
                          at<uint16_t>(plan, L.c_lo), at<uint16_t>(plan, L.c_h16), at<float>(plan, L.tnorm_blk),
                          plan->T, plan->Tpad, plan->k, plan->stream));
    plan->have_coeffs = true;
    return RBMF_OK;
}

rbmf_status rbmf_prepare_strain(rbmf_plan* plan, const float* x_dev, const float* inv_asd_dev, int32_t n_segments,
                                void* strain_out_dev) {
    if (!plan || !x_dev || !strain_out_dev) return RBMF_ERR_ARG;
    if (!plan->have_ws) return RBMF_ERR_STATE;
    if (n_segments < 1 || n_segments > plan->max_batch) return RBMF_ERR_ARG;
    if (((uintptr_t)x_dev % 8) != 0 || ((uintptr_t)strain_out_dev % 8) != 0) return RBMF_ERR_ARG;
    const Layout& L = plan->lay;
    CK(launch_r2c(x_dev, inv_asd_dev, at<float2>(plan, L.r2c_s), at<float2>(plan, L.r2c_z), (float2*)strain_out_dev,
                  at<float2>(plan, L.twF), plan->logN1 + plan->logN2, n_segments, plan->stream));
    return RBMF_OK;
}

rbmf_status rbmf_filter(rbmf_plan* plan, const void* strain_dev, float thr_stage1, float thr_stage2,
                        rbmf_trigger* out_dev, int64_t* n_out_dev) {
    return rbmf_filter_batch(plan, strain_dev, 1, thr_stage1, thr_stage2, out_dev, n_out_dev);
}

rbmf_status rbmf_filter_batch(rbmf_plan* plan, const void* strain_dev, int32_t n_segments, float thr_stage1,
                              float thr_stage2, rbmf_trigger* out_dev, int64_t* n_out_dev) {
    if (!plan || !strain_dev || !out_dev || !n_out_dev) return RBMF_ERR_ARG;
    if (!(thr_stage1 > 0.f) || !(thr_stage2 > 0.f)) return RBMF_ERR_ARG;
    if (n_segments < 1 || n_segments > plan->max_batch) return RBMF_ERR_ARG;
    if (!plan->have_ws || !plan->have_basis || !plan->have_coeffs) return RBMF_ERR_STATE;
    // every argument and state check comes before the first launch: a refused call leaves the plan's arrays untouched
    const bool by_templates = plan->stage1_route == RBMF_STAGE1_TEMPLATES;
    if (by_templates && n_segments != 1) return RBMF_ERR_UNSUPPORTED;
    if (by_templates && !plan->have_templates) return RBMF_ERR_STATE;
    const Layout& L = plan->lay;
    cudaStream_t st = plan->stream;
    const bool tm = plan->timing != 0;
    const int nb = n_segments;
    const int64_t Mtot = plan->M * nb;                       // bins of the whole batch
    const int64_t Mplane = plan->M * plan->max_batch;        // rows of the planes
    unsigned long long* counters = at<unsigned long long>(plan, L.counters);

    if (tm) {
        plan->ev_slot = (plan->ev_slot + 1) % kEvRing;
        ++plan->ev_calls;
        CK(cudaEventRecord(plan->ev[plan->ev_slot][0], st));
    }
    // counters + FFT scheduler words + per-bin histogram
    CK(cudaMemsetAsync(counters, 0, kCounterBytes + L.sched_bytes + (size_t)Mtot * 4, st));
    CK(launch_prep_strain((const float2*)strain_dev, at<float2>(plan, L.dsT), plan->logN1, plan->logN2,
                          (float)sqrt(2.0 / (double)plan->N), nb, st));

    // ---- kernel 1: a1-a3, one persistent launch over all (basis chunk, segment) pairs ----------------
    FftArgs a;
    memset(&a, 0, sizeof(a));
    a.basisP = at<float2>(plan, L.basisP); a.dsT = at<float2>(plan, L.dsT);
    a.tw1_a = at<float2>(plan, L.tw1_a); a.tw1_b = at<float2>(plan, L.tw1_b); a.twN = at<float2>(plan, L.twN);
    a.beta = at<float2>(plan, L.beta);
    a.plane_hi = at<uint16_t>(plan, L.bavg_hi); a.plane_lo = at<uint16_t>(plan, L.bavg_lo);
    a.sched = at<unsigned>(plan, L.sched);
    a.N = plan->N; a.M = (int)Mplane; a.Mseg = (int)plan->M; a.nb = nb;
    a.nchunk = plan->k / kFftC; a.w = plan->w; a.inv_w = 1.0f / (float)plan->w;
    const bool screen = plan->gemm_impl == RBMF_GEMM_SCREEN && !plan->diag_fp32_check;
    a.plane_fp16 = screen ? 1 : 0;
    // Batches run segment-major (every segment streams the basis from HBM again): keeping a basis chunk in L2 for the
    // other segments (chunk-major) displaces the in-place intermediate Y and measured 5-10 % slower per segment at
    // every size (Small B = 8: 0.74 vs 0.70 ms; Paper B = 4: 3.69 vs 3.37 ms) -- the kernel is not bound by that stream.
    a.seg_major = plan->diag_fft_chunk_major ? 0 : 1;
    {
        // Pass-1 lookahead: a chunk's pass 2 needs ALL of its pass-1 tiles, so enough pass-1 tiles of later chunks
        // must be queued to keep every consumer group (2 per SM) busy meanwhile -- about two tiles per group --,
        // limited by what Y (N x 32 bytes per chunk, lookahead + 1 chunks alive) may occupy in L2 (48 MB).
        const long long n1t = (1ll << plan->logN2) / fft_sub(plan->logN1);
        long long la = (4ll * plan->fft_grid + n1t - 1) / n1t;
        const long long cap = (48ll << 20) / ((long long)plan->N * kFftC * 8) - 1;
        if (la > cap) la = cap;
        if (la < 1) la = 1;
        if (plan->diag_fft_lookahead >= 1) la = plan->diag_fft_lookahead;
        a.lookahead = (int)la;
    }
    CK(launch_fft_tma(plan->tmY, a, plan->logN1, plan->logN2, plan->fft_grid, st));
    if (screen && !by_templates)
        CK(launch_bin_norm(at<uint16_t>(plan, L.bavg_hi), at<float>(plan, L.bin_norm), (int)Mtot, (int)Mplane,
                           (plan->k + 31) / 32, st));
    if (tm) CK(cudaEventRecord(plan->ev[plan->ev_slot][1], st));

    // ---- kernel 2: a4-a5 over the bins of all segments ------------------------------------------
    GemmArgs g;
    memset(&g, 0, sizeof(g));
    g.cand = at<rbmf_candidate>(plan, L.cand);
    g.bin_count = at<unsigned>(plan, L.bin_count);
    g.counters = counters;
    g.cand_cap = (unsigned long long)plan->max_cand;
    g.thr1_sq = thr_stage1 * thr_stage1;
    g.T = plan->T; g.M = (int)Mtot; g.k2 = 2 * plan->k;
    g.num_tb = plan->Tpad / kGemmTT;
    g.num_ib = (int)(Mtot / kGemmBM);
    {
        // template blocks per raster group: the group's coefficient tiles (256 rows x 2k values, one fp16 plane or bf16
        // hi + lo) stay L2-resident -- up to 48 MB of them -- while the beta^avg planes stream past once per group
        // (measured, Paper config: 32 blocks 2.05 ms, 64 blocks 2.03 ms, all 157 blocks 2.02 ms and a third of the
        // DRAM traffic)
        const size_t tile_bytes = (size_t)2 * kGemmTT * g.k2 * 2 * (screen ? 1 : 2);
        long long grp = (long long)((size_t)(48u << 20) / tile_bytes);
        g.group = (int)(grp < 8 ? 8 : (grp > g.num_tb ? g.num_tb : grp));
    }
    if (plan->diag_gemm_group >= 1) g.group = plan->diag_gemm_group;
    if (by_templates) {
        // the paper's fast first stage by templates (Eq. 10-12) in the place of the GEMM; exact fp32 candidates
        rbmf_status s1 = stage1_by_templates(plan, (const float2*)strain_dev, thr_stage1);
        if (s1 != RBMF_OK) return s1;
    } else if (screen) {
        // Bound of |R_fp16 - R| for the one-product fp16 screen (derivation: gemm_tcgen05.cu header): operand
        // rounding u = 2^-11 relative (+ eta = 2^-25 sqrt(2) absolute per complex value in the subnormal range), fp32
        // accumulation of the 2k exact products in the tensor core taken as (2k + 64) 2^-22 sqrt(2) relative to
        // ||a|| ||b|| (an assumption about the hardware's accumulator, checked against the oracle on the device by
        // tests/test_gpu_screen.py).  On top, kappa1 carries the fp32 rounding of the CONFIRM step in kernel 3 -- a
        // dot product of 2k real terms per component and the mean of w of them, gamma = (2k + w + 8) 2^-24 sqrt(2)
        // relative to ||a|| times the row norm, for which the bin norm stands in -- so that whatever the confirm
        // accepts, the screen has passed; `slack` covers the rounding of this threshold arithmetic itself.
        const double u = ldexp(1.0, -11), eta = ldexp(1.0, -25) * 1.4142135623730951;
        const double k = (double)plan->k;
        g.bin_norm = at<float>(plan, L.bin_norm);
        g.tnorm_blk = at<float>(plan, L.tnorm_blk);
        g.thr1 = thr_stage1;
        const double confirm = (2.0 * k + (double)plan->w + 8.0) * ldexp(1.0, -24) * 1.4142135623730951;
        g.kappa1 = (float)((2.0 * u + u * u + (2.0 * k + 64.0) * ldexp(1.0, -22) * 1.4142135623730951 + confirm) * 1.001);
        g.kappa2 = (float)(eta * sqrt(k) * 1.001);
        g.slack = 1e-4f;
        CK(launch_gemm_screen(plan->tmA_hi, plan->tmB_h16, plan->tmB_h16half,
                              plan->diag_single_cta ? 0 : plan->pair_clusters, g, plan->num_sms, st));
    } else if (!plan->diag_fp32_check) {
        CK(launch_gemm_tcgen05(plan->tmA_hi, plan->tmA_lo, plan->tmB_hi, plan->tmB_lo, g, plan->num_sms, st));
    } else {
        CK(launch_gemm_simt(at<uint16_t>(plan, L.bavg_hi), at<uint16_t>(plan, L.bavg_lo), at<uint16_t>(plan, L.c_hi),
                            at<uint16_t>(plan, L.c_lo), g, (int)Mplane, st));
    }
    if (tm) CK(cudaEventRecord(plan->ev[plan->ev_slot][2], st));

    // ---- kernel 3: a6 (candidates regrouped by bin; one warp per candidate where a bin's block is too large) ----
    Stage2Args s2;
    memset(&s2, 0, sizeof(s2));
    s2.cand = g.cand; s2.cs = at<float2>(plan, L.cs); s2.beta = at<float2>(plan, L.beta);
    s2.out = out_dev; s2.counters = counters;
    s2.trig_counter = plan->shared_trig_counter ? plan->shared_trig_counter : counters + 1;
    s2.template_offset = plan->template_offset;
    const bool confirm = screen && !by_templates;   // the list is the fp16 screen's superset: confirm in fp32
    s2.confirmed = at<rbmf_candidate>(plan, L.cand2); s2.thr1_sq = g.thr1_sq; s2.screen = confirm ? 1 : 0;
    s2.cand_cap = (unsigned long long)plan->max_cand;
    s2.trig_cap = plan->shared_trig_counter ? plan->shared_trig_cap : (unsigned long long)plan->max_trig;
    s2.thr2_sq = thr_stage2 * thr_stage2; s2.k = plan->k; s2.w = plan->w; s2.N = plan->N;
    s2.bin_count = g.bin_count; s2.bin_start = at<unsigned>(plan, L.bin_start); s2.items = at<int4>(plan, L.items);
    s2.sorted = at<rbmf_candidate>(plan, L.cand3);
    s2.Mseg = (int)plan->M; s2.Mtot = (int)Mtot; s2.seg_stride = (size_t)plan->N * plan->k;
    s2.smem_bytes = stage2_bybin_smem(plan->w, plan->k);
    if (s2.smem_bytes > 0 && !plan->diag_stage2_per_cand) CK(launch_stage2_bybin(s2, plan->num_sms, st));
    else CK(launch_stage2(s2, plan->num_sms, st));
    CK(cudaMemcpyAsync(n_out_dev, counters + 1, 8, cudaMemcpyDeviceToDevice, st));
    if (tm) CK(cudaEventRecord(plan->ev[plan->ev_slot][3], st));
    plan->filtered = true;
    plan->last_nb = nb;
    plan->last_impl = confirm ? (int)RBMF_GEMM_SCREEN : (int)RBMF_GEMM_TCGEN05;
    return RBMF_OK;
}

rbmf_status rbmf_plan_enable_template_routes(rbmf_plan* plan, int32_t slab) {
    if (!plan) return RBMF_ERR_ARG;
    if (plan->have_ws) return RBMF_ERR_STATE;
    if (slab < 0 || slab > 4 * kMaxChunks || (slab % kFftC) != 0) return RBMF_ERR_ARG;
    if (slab > 0 && (plan->w < 2 || 2 * plan->N / plan->w < 1024)) return RBMF_ERR_UNSUPPORTED;
    plan->tm_slab = slab;
    refresh(plan);
    return RBMF_OK;
}

rbmf_status rbmf_plan_set_stage1_route(rbmf_plan* plan, int32_t route) {
    if (!plan) return RBMF_ERR_ARG;
    if (route != RBMF_STAGE1_BASIS && route != RBMF_STAGE1_TEMPLATES) return RBMF_ERR_ARG;
    if (route == RBMF_STAGE1_TEMPLATES && plan->tm_slab == 0) return RBMF_ERR_STATE;
    plan->stage1_route = route;
    return RBMF_OK;
}

rbmf_status rbmf_set_templates(rbmf_plan* plan, const void* templates_dev, const float* sigma_dev) {
    if (!plan || !templates_dev) return RBMF_ERR_ARG;
    if (!plan->have_ws || plan->tm_slab == 0) return RBMF_ERR_STATE;
    CK(launch_tm_inv_sigma(sigma_dev, at<float>(plan, plan->lay.tm_isg), plan->T, plan->stream));
    plan->tm_templates = templates_dev;
    plan->have_templates = true;
    return RBMF_OK;
}

rbmf_status rbmf_filter_flat(rbmf_plan* plan, const void* strain_dev, float thr, rbmf_trigger* out_dev,
                             int64_t* n_out_dev) {
    if (!plan || !strain_dev || !out_dev || !n_out_dev || !(thr > 0.f)) return RBMF_ERR_ARG;
    if (!plan->have_ws || plan->tm_slab == 0 || !plan->have_templates) return RBMF_ERR_STATE;
    const Layout& L = plan->lay;
    const TmUnit& U = plan->tmF;
    cudaStream_t st = plan->stream;
    unsigned long long* counters = at<unsigned long long>(plan, L.counters);
    const bool tm = plan->timing != 0;
    if (tm) {
        plan->ev_slot = (plan->ev_slot + 1) % kEvRing;
        ++plan->ev_calls;
        CK(cudaEventRecord(plan->ev[plan->ev_slot][0], st));
    }
    CK(cudaMemsetAsync(counters, 0, kCounterBytes, st));
    CK(launch_prep_strain((const float2*)strain_dev, at<float2>(plan, U.dsT), U.logN1, U.logN2,
                          (float)sqrt(2.0 / (double)plan->N), 1, st));
    if (tm) { CK(cudaEventRecord(plan->ev[plan->ev_slot][1], st)); CK(cudaEventRecord(plan->ev[plan->ev_slot][2], st)); }
    for (int t0 = 0; t0 < plan->T; t0 += U.ncols) {
        CK(launch_layout_basis((const float2*)plan->tm_templates + (size_t)t0 * (size_t)(plan->N / 2 + 1),
                               at<float2>(plan, U.basisP), U.ncols, plan->N / 2 + 1, plan->j_low, U.logN1, U.logN2,
                               fft_sub(U.logN1), plan->T - t0, st));
        rbmf_status s = run_tm_unit(plan, U);
        if (s != RBMF_OK) return s;
        CK(launch_tm_scan(at<float2>(plan, U.beta), U.N, 1, (int)plan->N, at<float>(plan, L.tm_isg), t0, plan->T,
                          U.ncols, thr * thr, out_dev, counters + 1, (unsigned long long)plan->max_trig, nullptr, st));
    }
    CK(cudaMemcpyAsync(n_out_dev, counters + 1, 8, cudaMemcpyDeviceToDevice, st));
    if (tm) CK(cudaEventRecord(plan->ev[plan->ev_slot][3], st));
    plan->filtered = true;
    plan->last_nb = 1;
    plan->last_impl = RBMF_GEMM_TCGEN05;   // counters[0] (unused here: 0 candidates) is the final candidate count
    return RBMF_OK;
}

rbmf_status rbmf_get_counts(rbmf_plan* plan, int64_t* n_candidates, int64_t* n_triggers) {
    if (!plan) return RBMF_ERR_ARG;
    if (!plan->filtered) return RBMF_ERR_STATE;
    unsigned long long h[3] = {0, 0, 0};
    CK(cudaMemcpyAsync(h, plan->ws + plan->lay.counters, 24, cudaMemcpyDeviceToHost, plan->stream));
    CK(cudaStreamSynchronize(plan->stream));
    // screen mode: h[0] counts the screened superset, h[2] the candidates confirmed at fp32 accuracy
    const bool screen = plan->last_impl == RBMF_GEMM_SCREEN;
    if (n_candidates) *n_candidates = (int64_t)(screen ? h[2] : h[0]);
    if (n_triggers) *n_triggers = (int64_t)h[1];
    if ((int64_t)h[0] > plan->max_cand || (int64_t)h[1] > plan->max_trig) return RBMF_ERR_OVERFLOW;
    return RBMF_OK;
}

rbmf_status rbmf_get_screened_count(rbmf_plan* plan, int64_t* n_screened) {
    if (!plan || !n_screened) return RBMF_ERR_ARG;
    if (!plan->filtered) return RBMF_ERR_STATE;
    unsigned long long h = 0;
    CK(cudaMemcpyAsync(&h, plan->ws + plan->lay.counters, 8, cudaMemcpyDeviceToHost, plan->stream));
    CK(cudaStreamSynchronize(plan->stream));
    *n_screened = (int64_t)h;
    return RBMF_OK;
}

rbmf_status rbmf_diag_set(rbmf_plan* plan, int32_t option, int32_t value) {
    if (!plan) return RBMF_ERR_ARG;
    switch (option) {
        case RBMF_DIAG_STAGE1_FP32_CHECK: plan->diag_fp32_check = value ? 1 : 0; return RBMF_OK;
        case RBMF_DIAG_SINGLE_CTA_SCREEN: plan->diag_single_cta = value ? 1 : 0; return RBMF_OK;
        case RBMF_DIAG_STAGE2_PER_CANDIDATE: plan->diag_stage2_per_cand = value ? 1 : 0; return RBMF_OK;
        case RBMF_DIAG_FFT_CHUNK_MAJOR: plan->diag_fft_chunk_major = value ? 1 : 0; return RBMF_OK;
        case RBMF_DIAG_FFT_LOOKAHEAD:
            if (value < 0 || value > kMaxChunks) return RBMF_ERR_ARG;
            plan->diag_fft_lookahead = value;
            return RBMF_OK;
        case RBMF_DIAG_GEMM_GROUP:
            if (value < 0) return RBMF_ERR_ARG;
            plan->diag_gemm_group = value;
            return RBMF_OK;
        default: return RBMF_ERR_ARG;
    }
}

rbmf_status rbmf_get_candidates(rbmf_plan* plan, rbmf_candidate* out_host, int64_t capacity, int64_t* n_out) {
    if (!plan || !out_host || !n_out || capacity < 0) return RBMF_ERR_ARG;
    int64_t nc = 0, nt = 0;
    rbmf_status s = rbmf_get_counts(plan, &nc, &nt);
    if (s != RBMF_OK && s != RBMF_ERR_OVERFLOW) return s;
    *n_out = nc;
    int64_t n = nc < plan->max_cand ? nc : plan->max_cand;
    if (n > capacity) n = capacity;
    if (n > 0) {
        const size_t off = plan->last_impl == RBMF_GEMM_SCREEN ? plan->lay.cand2 : plan->lay.cand;
        CK(cudaMemcpyAsync(out_host, plan->ws + off, (size_t)n * sizeof(rbmf_candidate),
                           cudaMemcpyDeviceToHost, plan->stream));
        CK(cudaStreamSynchronize(plan->stream));
    }
    return s;
}

rbmf_status rbmf_filter_host(rbmf_plan* plan, const void* strain_host, float thr_stage1, float thr_stage2,
                             rbmf_trigger* out_host, int64_t capacity_out, int64_t* n_out_host) {
    return rbmf_filter_batch_host(plan, strain_host, 1, thr_stage1, thr_stage2, out_host, capacity_out, n_out_host);
}

rbmf_status rbmf_filter_batch_host(rbmf_plan* plan, const void* strain_host, int32_t n_segments, float thr_stage1,
                                   float thr_stage2, rbmf_trigger* out_host, int64_t capacity_out,
                                   int64_t* n_out_host) {
    if (!plan || !strain_host || !out_host || !n_out_host || capacity_out < 1) return RBMF_ERR_ARG;
    if (!plan->have_ws || !plan->have_basis || !plan->have_coeffs) return RBMF_ERR_STATE;
    if (n_segments < 1 || n_segments > plan->max_batch) return RBMF_ERR_ARG;
    if (capacity_out > plan->max_trig) capacity_out = plan->max_trig;
    const Layout& L = plan->lay;
    const size_t strain_bytes = (size_t)n_segments * (size_t)(plan->N / 2 + 1) * 8;
    uint8_t* strain_dev = plan->ws + L.strain_stage;
    rbmf_trigger* trig_dev = (rbmf_trigger*)(plan->ws + L.trig_stage);
    int64_t* n_dev = (int64_t*)(plan->ws + L.counters + 64);   // counter word 8
    CK(cudaMemcpyAsync(strain_dev, strain_host, strain_bytes, cudaMemcpyHostToDevice, plan->stream));
    rbmf_status s = rbmf_filter_batch(plan, strain_dev, n_segments, thr_stage1, thr_stage2, trig_dev, n_dev);
    if (s != RBMF_OK) return s;
    int64_t nc = 0, nt = 0;
    s = rbmf_get_counts(plan, &nc, &nt);
    if (s != RBMF_OK && s != RBMF_ERR_OVERFLOW) return s;
    *n_out_host = nt;
    int64_t n = nt < capacity_out ? nt : capacity_out;
    if (n > 0) {
        CK(cudaMemcpyAsync(out_host, trig_dev, (size_t)n * sizeof(rbmf_trigger), cudaMemcpyDeviceToHost,
                           plan->stream));
        CK(cudaStreamSynchronize(plan->stream));
    }
    return s;
}

rbmf_status rbmf_get_internal(rbmf_plan* plan, int32_t which, const void** dev_ptr, size_t* bytes) {
    if (!plan || !dev_ptr || !bytes) return RBMF_ERR_ARG;
    if (!plan->have_ws) return RBMF_ERR_STATE;
    const Layout& L = plan->lay;
    switch (which) {
        case 0: *dev_ptr = plan->ws + L.beta; *bytes = (size_t)plan->max_batch * plan->N * plan->k * 8; break;
        case 1: *dev_ptr = plan->ws + L.bavg_hi; *bytes = L.plane_bytes; break;
        case 2: *dev_ptr = plan->ws + L.bavg_lo; *bytes = L.plane_bytes; break;
        case 3: *dev_ptr = plan->ws + L.cand; *bytes = (size_t)plan->max_cand * sizeof(rbmf_candidate); break;
        case 4: *dev_ptr = plan->ws + L.bin_norm; *bytes = (size_t)plan->M * plan->max_batch * 4; break;
        case 5: *dev_ptr = plan->ws + L.tnorm_blk; *bytes = (size_t)(plan->Tpad / kGemmTT) * 4; break;
        case 6:
            *dev_ptr = plan->ws + (plan->last_impl == RBMF_GEMM_SCREEN ? L.cand2 : L.cand);
            *bytes = (size_t)plan->max_cand * sizeof(rbmf_candidate);
            break;
        default: return RBMF_ERR_ARG;
    }
    return RBMF_OK;
}

rbmf_status rbmf_plan_set_timing(rbmf_plan* plan, int32_t enabled) {
    if (!plan) return RBMF_ERR_ARG;
    plan->timing = enabled ? 1 : 0;
    plan->ev_calls = 0;   // the history starts over
    return RBMF_OK;
}

rbmf_status rbmf_get_stage_ms_history(rbmf_plan* plan, int32_t calls_back, float ms[4]) {
    if (!plan || !ms || calls_back < 0 || calls_back >= kEvRing) return RBMF_ERR_ARG;
    if (!plan->filtered || !plan->timing || !plan->have_events) return RBMF_ERR_STATE;
    if ((long long)calls_back >= plan->ev_calls) return RBMF_ERR_STATE;   // fewer timed calls than that so far
    cudaEvent_t* ev = plan->ev[(plan->ev_slot - calls_back + kEvRing) % kEvRing];
    CK(cudaEventSynchronize(plan->ev[plan->ev_slot][3]));
    CK(cudaEventElapsedTime(&ms[0], ev[0], ev[1]));
    CK(cudaEventElapsedTime(&ms[1], ev[1], ev[2]));
    CK(cudaEventElapsedTime(&ms[2], ev[2], ev[3]));
    CK(cudaEventElapsedTime(&ms[3], ev[0], ev[3]));
    return RBMF_OK;
}

rbmf_status rbmf_get_stage_ms(rbmf_plan* plan, float ms[4]) { return rbmf_get_stage_ms_history(plan, 0, ms); }

rbmf_status rbmf_launches_per_filter(const rbmf_plan* plan, int32_t* n) {
    if (!plan || !n) return RBMF_ERR_ARG;
    // prep_strain + fused FFT + (screen: bin norms) + GEMM + stage 2 (by bin: alloc, scatter, score)
    const int s2 = (stage2_bybin_smem(plan->w, plan->k) > 0 && !plan->diag_stage2_per_cand) ? 3 : 1;
    *n = ((plan->gemm_impl == RBMF_GEMM_SCREEN && !plan->diag_fp32_check) ? 4 : 3) + s2;
    return RBMF_OK;
}

rbmf_status rbmf_plan_destroy(rbmf_plan* plan) {
    if (!plan) return RBMF_ERR_ARG;
    if (plan->have_events)
        for (int r = 0; r < kEvRing; ++r)
            for (int i = 0; i < 4; ++i) cudaEventDestroy(plan->ev[r][i]);
    delete plan;
    return RBMF_OK;
}

const char* rbmf_status_string(rbmf_status status) {
    switch (status) {
        case RBMF_OK: return "ok";
        case RBMF_ERR_ARG: return "invalid argument";
        case RBMF_ERR_STATE: return "call order: workspace, basis or coefficients not set";
        case RBMF_ERR_CUDA: return "CUDA error (see rbmf_last_cuda_error)";
        case RBMF_ERR_OVERFLOW: return "candidate or trigger capacity exceeded; lists truncated";
        case RBMF_ERR_UNSUPPORTED: return "unsupported size or device";
        default: return "unknown status";
    }
}

int32_t rbmf_last_cuda_error(const rbmf_plan* plan) { return plan ? plan->last_cuda : 0; }

// ---- preparation on the GPU ---------------------------------------------------
namespace {
bool prep_args_ok(int64_t N, double fs, double f_low, int* j_low, int64_t* n_half) {
    if (N < 64 || (N & (N - 1)) != 0 || N > (int64_t(1) << 24)) return false;
    if (!(fs > 0.0) || !(f_low > 0.0) || !(f_low < fs / 2)) return false;
    *n_half = N / 2;
    *j_low = (int)ceil(f_low * (double)N / fs - 1e-12);
    return *j_low < *n_half;
}
}  // namespace

rbmf_status rbmf_prepare_basis_workspace_bytes(int32_t n_templates, int32_t k, size_t* bytes) {
    if (!bytes || n_templates < 1 || k < 1 || k > n_templates || n_templates > 32768) return RBMF_ERR_ARG;
    *bytes = prep_basis_workspace_bytes(n_templates, k);
    return RBMF_OK;
}

rbmf_status rbmf_prepare_basis(const void* templates_dev, int32_t n_templates, int64_t N, double fs, double f_low,
                               int32_t k, int32_t iterations, uint64_t seed, void* workspace_dev, size_t workspace_bytes,
                               void* basis_out_dev, float* eig_out_dev, void* cuda_stream) {
    int j_low = 0;
    int64_t n_half = 0;
    if (!templates_dev || !workspace_dev || !basis_out_dev || !prep_args_ok(N, fs, f_low, &j_low, &n_half)) return RBMF_ERR_ARG;
    if (n_templates < 1 || n_templates > 32768 || k < 1 || k > n_templates || k > 1024 || iterations < 1 || iterations > 1000)
        return RBMF_ERR_ARG;
    if (((uintptr_t)workspace_dev % 16) != 0 || workspace_bytes < prep_basis_workspace_bytes(n_templates, k)) return RBMF_ERR_ARG;
    cudaError_t e = launch_prep_basis((const float2*)templates_dev, n_templates, N / 2 + 1, j_low, n_half, k, iterations,
                                      (unsigned long long)seed, workspace_dev, (float2*)basis_out_dev, eig_out_dev,
                                      (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? RBMF_OK : RBMF_ERR_CUDA;
}

rbmf_status rbmf_prepare_coeffs(const void* templates_dev, int32_t n_templates, const void* basis_dev, int32_t k,
                                int64_t N, double fs, double f_low, void* coeffs_out_dev, float* sigma_out_dev,
                                void* cuda_stream) {
    int j_low = 0;
    int64_t n_half = 0;
    if (!templates_dev || !basis_dev || !coeffs_out_dev || !prep_args_ok(N, fs, f_low, &j_low, &n_half)) return RBMF_ERR_ARG;
    if (n_templates < 1 || n_templates > (1 << 24) || k < 1 || k > 1024) return RBMF_ERR_ARG;
    cudaError_t e = launch_prep_coeffs_from_templates((const float2*)templates_dev, n_templates, (const float2*)basis_dev, k,
                                                      N / 2 + 1, j_low, n_half, (float2*)coeffs_out_dev, sigma_out_dev,
                                                      (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? RBMF_OK : RBMF_ERR_CUDA;
}

// ---- bank sets: many sub-banks against one strain (Table I) ------------------------
struct rbmf_bankset {
    int n;
    rbmf_plan** plans;
    int* order;          // launch order: most expensive sub-bank first
    int* offsets;        // template id base of each sub-bank
    int nstreams;
    cudaStream_t streams[4];
    cudaEvent_t fork, join[4];
    cudaEvent_t plan_ready;   // re-recorded per sub-bank on the plan's own stream: its set-up work precedes the filter
    cudaStream_t last_stream;
    unsigned long long* last_counter;
    bool filtered;
};

rbmf_status rbmf_bankset_create(rbmf_bankset** out, rbmf_plan* const* plans, int32_t n_plans) {
    if (!out) return RBMF_ERR_ARG;
    *out = nullptr;
    if (!plans || n_plans < 1 || n_plans > 4096) return RBMF_ERR_ARG;
    int64_t total_T = 0;
    for (int i = 0; i < n_plans; ++i) {
        const rbmf_plan* p = plans[i];
        if (!p) return RBMF_ERR_ARG;
        if (!p->have_ws || !p->have_basis || !p->have_coeffs) return RBMF_ERR_STATE;
        if (p->N != plans[0]->N || p->fs != plans[0]->fs || p->f_low != plans[0]->f_low) return RBMF_ERR_ARG;
        for (int j = 0; j < i; ++j)
            if (plans[j] == p) return RBMF_ERR_ARG;
        total_T += p->T;
    }
    if (total_T > (int64_t(1) << 31) - 1) return RBMF_ERR_ARG;
    rbmf_bankset* b = new (std::nothrow) rbmf_bankset;
    if (!b) return RBMF_ERR_ARG;
    memset(b, 0, sizeof(*b));
    b->n = n_plans;
    b->plans = new (std::nothrow) rbmf_plan*[n_plans];
    b->order = new (std::nothrow) int[n_plans];
    b->offsets = new (std::nothrow) int[n_plans];
    if (!b->plans || !b->order || !b->offsets) { delete[] b->plans; delete[] b->order; delete[] b->offsets; delete b; return RBMF_ERR_ARG; }
    int off = 0;
    for (int i = 0; i < n_plans; ++i) { b->plans[i] = plans[i]; b->order[i] = i; b->offsets[i] = off; off += plans[i]->T; }
    // longest first: the cost of a sub-bank is dominated by its reconstruction, 8 T k N / w flops
    auto cost = [&](int i) { const rbmf_plan* p = b->plans[i]; return (double)p->T * p->k * (double)p->M; };
    for (int i = 1; i < n_plans; ++i) {
        const int v = b->order[i];
        int j = i - 1;
        while (j >= 0 && cost(b->order[j]) < cost(v)) { b->order[j + 1] = b->order[j]; --j; }
        b->order[j + 1] = v;
    }
    b->nstreams = n_plans < 4 ? n_plans : 4;
    rbmf_plan* plan = plans[0];   // for CK's error slot
    cudaError_t e = cudaEventCreateWithFlags(&b->fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&b->plan_ready, cudaEventDisableTiming);
    for (int i = 0; i < b->nstreams && e == cudaSuccess; ++i) {
        e = cudaStreamCreateWithFlags(&b->streams[i], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&b->join[i], cudaEventDisableTiming);
    }
    if (e != cudaSuccess) { rbmf_bankset_destroy(b); return cuda_fail(plan, e); }
    *out = b;
    return RBMF_OK;
}

rbmf_status rbmf_bankset_filter(rbmf_bankset* bs, const void* strain_dev, float thr_stage1, float thr_stage2,
                                rbmf_trigger* out_dev, int64_t max_triggers, int64_t* n_out_dev, void* cuda_stream) {
    if (!bs || !strain_dev || !out_dev || !n_out_dev || max_triggers < 1) return RBMF_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    rbmf_plan* plan = bs->plans[0];
    CK(cudaMemsetAsync(n_out_dev, 0, 8, st));
    CK(cudaEventRecord(bs->fork, st));
    for (int i = 0; i < bs->nstreams; ++i) CK(cudaStreamWaitEvent(bs->streams[i], bs->fork, 0));
    rbmf_status result = RBMF_OK;
    for (int q = 0; q < bs->n && result == RBMF_OK; ++q) {
        rbmf_plan* p = bs->plans[bs->order[q]];
        cudaStream_t saved = p->stream;
        // what the caller has enqueued on the plan's own stream (rbmf_set_basis / rbmf_set_coeffs, an earlier
        // rbmf_filter) comes first: the internal streams are non-blocking and ordered against `cuda_stream` only
        CK(cudaEventRecord(bs->plan_ready, saved));
        CK(cudaStreamWaitEvent(bs->streams[q % bs->nstreams], bs->plan_ready, 0));
        p->stream = bs->streams[q % bs->nstreams];
        p->shared_trig_counter = (unsigned long long*)n_out_dev;
        p->shared_trig_cap = (unsigned long long)max_triggers;
        p->template_offset = bs->offsets[bs->order[q]];
        // the plan's own trigger count lands in its counter word 9 (word 8 belongs to rbmf_filter_host)
        result = rbmf_filter(p, strain_dev, thr_stage1, thr_stage2, out_dev,
                             (int64_t*)(p->ws + p->lay.counters + 72));
        p->stream = saved;
        p->shared_trig_counter = nullptr;
        p->template_offset = 0;
    }
    for (int i = 0; i < bs->nstreams; ++i) {
        CK(cudaEventRecord(bs->join[i], bs->streams[i]));
        CK(cudaStreamWaitEvent(st, bs->join[i], 0));
    }
    bs->last_stream = st;
    bs->last_counter = (unsigned long long*)n_out_dev;
    bs->filtered = result == RBMF_OK;
    return result;
}

rbmf_status rbmf_bankset_get_counts(rbmf_bankset* bs, int64_t* n_candidates, int64_t* n_triggers, int64_t* n_total) {
    if (!bs) return RBMF_ERR_ARG;
    if (!bs->filtered) return RBMF_ERR_STATE;
    rbmf_plan* plan = bs->plans[0];
    CK(cudaStreamSynchronize(bs->last_stream));
    rbmf_status result = RBMF_OK;
    unsigned long long total = 0;
    for (int i = 0; i < bs->n; ++i) {
        rbmf_plan* p = bs->plans[i];
        unsigned long long h[3] = {0, 0, 0};
        CK(cudaMemcpy(h, p->ws + p->lay.counters, 24, cudaMemcpyDeviceToHost));
        if (n_candidates) n_candidates[i] = (int64_t)(p->last_impl == RBMF_GEMM_SCREEN ? h[2] : h[0]);
        if (n_triggers) n_triggers[i] = (int64_t)h[1];
        total += h[1];
        if ((int64_t)h[0] > p->max_cand) result = RBMF_ERR_OVERFLOW;
    }
    unsigned long long shared = 0;
    CK(cudaMemcpy(&shared, bs->last_counter, 8, cudaMemcpyDeviceToHost));
    if (n_total) *n_total = (int64_t)shared;
    if (shared != total) { plan->last_cuda = -2; return RBMF_ERR_CUDA; }   // cannot happen: both count the same appends
    return result;
}

rbmf_status rbmf_bankset_destroy(rbmf_bankset* bs) {
    if (!bs) return RBMF_ERR_ARG;
    for (int i = 0; i < bs->nstreams; ++i) {
        if (bs->streams[i]) { cudaStreamSynchronize(bs->streams[i]); cudaStreamDestroy(bs->streams[i]); }
        if (bs->join[i]) cudaEventDestroy(bs->join[i]);
    }
    if (bs->fork) cudaEventDestroy(bs->fork);
    if (bs->plan_ready) cudaEventDestroy(bs->plan_ready);
    delete[] bs->plans; delete[] bs->order; delete[] bs->offsets;
    delete bs;
    return RBMF_OK;
}

}  // extern "C"
