// Kernel 2 (steps a4-a5): stage-1 template reconstruction as a split-precision complex GEMM on the 5th-generation
// tensor cores, with normalisation, threshold and candidate compaction fused into the TMEM epilogue, so the
// T x N/w averaged-SNR matrix never reaches HBM (Eq. 7 :90).
//
// Real formulation.  With c_tk = a + i b and beta^avg_k[i] = x + i y,
//     Re R_t[i] = sum_k (a x + b y)/sigma_t,   Im R_t[i] = sum_k (a y - b x)/sigma_t,
// i.e. two real dot products of length 2k between the time-bin row (x_0, y_0, x_1, y_1, ...) and the template rows
// "re" = (a_0, b_0, ...)/sigma and "im" = (-b_0, a_0, ...)/sigma (built by prep_coeffs_kernel).
//
// Tile: D[128 time bins x 256] = A[128 x 2k] * B[256 x 2k]^T, where the 256 B rows are the 128 "re" rows followed by
// the 128 "im" rows of one block of 128 templates.  Time bins sit on the UMMA M dimension (TMEM lanes), templates on N
// (TMEM columns): thread <-> time bin, and Re/Im of (bin, template) are columns c and 128 + c of the SAME lane, so
// the epilogue needs no shuffles.  One N = 256 instruction per product keeps shared-memory operand traffic at
// (4 KB A + 8 KB B) per 128 tensor-pipe cycles.
//
// Split precision (bf16x3): every fp32 operand value v is stored as hi = bf16(v), lo = bf16(v - hi); the product is
// accumulated in fp32 as  A_hi B_hi + A_hi B_lo + A_lo B_hi  (the lo*lo term, ~2^-16 relative, is dropped).
//
// Screen mode (MODE 1, RBMF_GEMM_SCREEN, the default).  ONE product with both operands rounded once to fp16, and the
// threshold of every (time bin i, template block) lowered by a bound of the error this can cause, so that the hit list
// is a superset of the true candidates; kernel 3 repeats the test in fp32 (see stage2_kernels.cu).  With a = c_t/sigma_t,
// b = beta^avg[i] (the fp32 values), u = 2^-11 and eta = sqrt(2) 2^-25 (fp16 subnormal range):
//     |delta a_k| <= u |a_k| + eta,  |delta b_k| <= u |b_k| + eta        (each complex component rounded to nearest)
//     |R_16 - R| <= (2u + u^2) ||a|| ||b|| + eta sqrt(k) (||a|| + ||b||)                       (Cauchy-Schwarz)
//                   + (2k + 64) 2^-22 sqrt(2) ||a|| ||b||        (fp32 accumulation of the 2k exact fp16 products)
// ||b|| comes from bin_norm_kernel (GemmArgs::bin_norm, inflated for the rounding of the plane it reads), ||a|| as the
// maximum over the tile's 128 templates (GemmArgs::tnorm_blk); kappa1, kappa2, slack are set in rbmf_api.cu.
//
// Warp roles (192 threads): warp 0 = TMA producer, warp 1 = TMEM allocator + single-thread tcgen05.mma issuer,
// warps 2-5 = epilogue (one TMEM lane quadrant each).  Two TMEM accumulator buffers (2 x 256 columns) let the epilogue
// of tile n overlap the main loop of tile n+1.  The kernel is persistent: grid = #SMs, static round-robin over tiles in
// an order that keeps a group of template blocks L2-resident while time-bin blocks stream.
#include <cuda_bf16.h>

#include "rbmf_internal.h"

namespace rbmf {

namespace {

constexpr int BM = kGemmBM;            // 128 time bins
constexpr int BN = 2 * kGemmTT;        // 256 = 128 templates x {re, im}
constexpr int BK = kGemmBK;            // 64 bf16 = 128 B
constexpr int UMMA_K = 16;
constexpr uint32_t A_BYTES = BM * BK * 2;                     // 16 KB per plane
constexpr uint32_t B_BYTES = BN * BK * 2;                     // 32 KB per plane
// MODE 0 (bf16x3): planes A_hi, A_lo, B_hi, B_lo = 96 KB per stage, 2 stages.
// MODE 1 (fp16 screen): one A and one B plane = 48 KB per stage, 4 stages.
template <int MODE> struct ModeCfg {
    static constexpr int PLANES = MODE == 0 ? 2 : 1;
    static constexpr int STAGES = MODE == 0 ? 2 : 4;
    static constexpr uint32_t STAGE_BYTES = PLANES * (A_BYTES + B_BYTES);
    static constexpr uint32_t SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*align*/ + 256 /*barriers*/;
};
constexpr uint32_t TMEM_COLS = 512;
constexpr int NUM_THREADS = 192;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(bar), "r"(parity)
            : "memory");
    } while (!done);
}

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(x), "r"(y)
        : "memory");
}

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(x), "r"(y), "r"(z)
        : "memory");
}

// K-major operand tile in shared memory, 128-byte rows, SWIZZLE_128B: 8-row groups are 1024 B apart (SBO);
// descriptor version 1 (sm_100), layout type 2 (SWIZZLE_128B).  Advancing along K by 16 bf16 = +32 B on the start
// address (the hardware applies the XOR swizzle on the absolute shared-memory address bits).
__device__ __forceinline__ uint64_t make_smem_desc(uint32_t addr) {
    uint64_t d = 0;
    d |= (uint64_t)((addr & 0x3FFFFu) >> 4);          // start address,        bits [0,14)
    d |= (uint64_t)1 << 16;                           // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024u >> 4) << 32;                // stride byte offset,   bits [32,46)
    d |= (uint64_t)1 << 46;                           // descriptor version
    d |= (uint64_t)2 << 61;                           // SWIZZLE_128B
    return d;
}

// kind::f16 instruction descriptors: D = F32, both operands K-major, N = 256, M = 128; A = B = BF16 (format 1) for
// the bf16x3 products, A = B = F16 (format 0) for the screen.
constexpr uint32_t kInstrDescF16 = (1u << 4) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
constexpr uint32_t kInstrDescBF16 = kInstrDescF16 | (1u << 7) | (1u << 10);

template <uint32_t IDESC>
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
        "l"(adesc), "l"(bdesc), "n"(IDESC), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Tile order: groups of `group` template blocks; inside a group, time-bin blocks outer, template blocks inner.
__device__ __forceinline__ void decode_tile(const GemmArgs& g, int tile, int& ib, int& tb) {
    const int per_group = g.group * g.num_ib;
    const int grp = tile / per_group;
    const int rem = tile - grp * per_group;
    const int tb0 = grp * g.group;
    const int gsz = min(g.group, g.num_tb - tb0);
    ib = rem / gsz;
    tb = tb0 + rem % gsz;
}

__device__ __forceinline__ int num_tiles(const GemmArgs& g) { return g.num_tb * g.num_ib; }

// Epilogue of one 128-bin x 128-template tile for one warp (its 32 TMEM lanes = 32 time bins).
// Pass 1 (every tile): |R|^2 against the threshold of this bin -- two packed fp32x2 ops and one max per two values --
// and one warp vote per 32 templates; the per-value hit masks are built only where the vote fired.
// Pass 2 (only if something hit): ONE atomicAdd per warp and tile reserves the list space for all its hits (a loud
// injection fires in thousands of tiles at once: per-column atomics on the single counter serialise in L2), then the
// chunks that hit are read from TMEM again and written out.
__device__ __forceinline__ void epilogue_tile(const GemmArgs& g, uint32_t taddr, int bin, int tb, int lane,
                                              float thr_sq) {
    constexpr int NCH = kGemmTT / 32;
    uint32_t mask[NCH];
    bool any = false;
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        uint32_t re[32], im[32];
        tmem_ld32(taddr + ch * 32, re);
        tmem_ld32(taddr + kGemmTT + ch * 32, im);
        tmem_ld_wait();
        // NaN (an fp16 overflow upstream) must pass the screen: fmaxf drops NaN operands, so the plain sum of the
        // squares is tracked too -- it stays NaN or inf if anything was.
        float vmax = 0.f, vsum = 0.f;
#pragma unroll
        for (int j = 0; j < 32; j += 2) {
            unsigned long long xx, yy, m2;
            asm("mov.b64 %0, {%1, %2};" : "=l"(xx) : "r"(re[j]), "r"(re[j + 1]));
            asm("mov.b64 %0, {%1, %2};" : "=l"(yy) : "r"(im[j]), "r"(im[j + 1]));
            asm("mul.rn.f32x2 %0, %1, %1;" : "=l"(m2) : "l"(yy));
            asm("fma.rn.f32x2 %0, %1, %1, %2;" : "=l"(m2) : "l"(xx), "l"(m2));
            float m0, m1;
            asm("mov.b64 {%0, %1}, %2;" : "=f"(m0), "=f"(m1) : "l"(m2));
            vmax = fmaxf(vmax, fmaxf(m0, m1));
            vsum += m0 + m1;
        }
        const bool maybe = bin < g.M && !(vmax < thr_sq && vsum < 3.0e38f);
        uint32_t m = 0;
        if (__any_sync(0xffffffffu, maybe)) {
#pragma unroll
            for (int j = 0; j < 32; ++j) {
                const float x = __uint_as_float(re[j]), y = __uint_as_float(im[j]);
                const bool hit = !(fmaf(x, x, y * y) < thr_sq) && (tb * kGemmTT + ch * 32 + j) < g.T;
                m |= (hit ? 1u : 0u) << j;
            }
            if (bin >= g.M) m = 0;
        }
        mask[ch] = m;
        any |= m != 0;
    }
    if (!__any_sync(0xffffffffu, any)) return;

    // ---- rare path: reserve, then write ------------------------------------------------------------------------
    int cnt = 0;
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) cnt += __popc(mask[ch]);
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(g.counters, (unsigned long long)total);
    base = __shfl_sync(0xffffffffu, base, 0);
    unsigned long long idx = base + (unsigned long long)(incl - cnt);
    if (cnt > 0 && idx < g.cand_cap) {
        // histogram of the entries actually written, per bin: stage 2 regroups the list by bin (stage2_bybin.cu)
        const unsigned long long room = g.cand_cap - idx;
        atomicAdd(g.bin_count + bin, (unsigned)(room < (unsigned long long)cnt ? room : (unsigned long long)cnt));
    }
#pragma unroll 1
    for (int ch = 0; ch < NCH; ++ch) {
        const uint32_t m = mask[ch];
        if (__ballot_sync(0xffffffffu, m != 0) == 0) continue;
        uint32_t re[32], im[32];
        tmem_ld32(taddr + ch * 32, re);
        tmem_ld32(taddr + kGemmTT + ch * 32, im);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            if ((m >> j) & 1u) {
                if (idx < g.cand_cap) {
                    rbmf_candidate cd;
                    cd.template_id = tb * kGemmTT + ch * 32 + j;
                    cd.bin_index = bin;
                    cd.avg_re = __uint_as_float(re[j]);
                    cd.avg_im = __uint_as_float(im[j]);
                    g.cand[idx] = cd;
                }
                ++idx;
            }
        }
    }
}

}  // namespace

template <int MODE>
__global__ void __launch_bounds__(NUM_THREADS, 1)
gemm_tcgen05_kernel(const __grid_constant__ CUtensorMap tmA_hi, const __grid_constant__ CUtensorMap tmA_lo,
                    const __grid_constant__ CUtensorMap tmB_hi, const __grid_constant__ CUtensorMap tmB_lo,
                    const GemmArgs g) {
    constexpr int STAGES = ModeCfg<MODE>::STAGES;
    constexpr uint32_t STAGE_BYTES = ModeCfg<MODE>::STAGE_BYTES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;
    // barrier slots (8 B each): full[STAGES], empty[STAGES], tmem_full[2], tmem_empty[2]; then the TMEM pointer
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + 2 + b); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA_hi) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA_lo) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB_hi) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB_lo) : "memory");
        for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "n"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    const int ntiles = num_tiles(g);
    const int num_kb = (g.k2 + BK - 1) / BK;   // a ragged last block is zero-filled by TMA (k2 = 32 when k = 16)

    if (warp == 0) {
        // ================================ TMA producer ================================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
                int ib, tb;
                decode_tile(g, tile, ib, tb);
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sbase = smem_base + stage * STAGE_BYTES;
                    mbar_expect_tx(full_bar(stage), STAGE_BYTES);
                    // beta^avg planes are K-block major, [kb][bin][64]: one box = 16 KB contiguous
                    if (MODE == 0) {
                        tma_load_3d(sbase, &tmA_hi, full_bar(stage), 0, ib * BM, kb);
                        tma_load_3d(sbase + A_BYTES, &tmA_lo, full_bar(stage), 0, ib * BM, kb);
                        tma_load_2d(sbase + 2 * A_BYTES, &tmB_hi, full_bar(stage), kb * BK, tb * BN);
                        tma_load_2d(sbase + 2 * A_BYTES + B_BYTES, &tmB_lo, full_bar(stage), kb * BK, tb * BN);
                    } else {
                        tma_load_3d(sbase, &tmA_hi, full_bar(stage), 0, ib * BM, kb);
                        tma_load_2d(sbase + A_BYTES, &tmB_hi, full_bar(stage), kb * BK, tb * BN);
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ================================ MMA issuer ==================================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            int it = 0;
            for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
                const int buf = it & 1;
                mbar_wait(tempty_bar(buf), ((uint32_t)(it >> 1) & 1u) ^ 1u);   // epilogue has drained this buffer
                tc_fence_after();
                const uint32_t tmem_d = tmem_base + (uint32_t)(buf * BN);
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sbase = smem_base + stage * STAGE_BYTES;
#pragma unroll
                    for (int k4 = 0; k4 < BK / UMMA_K; ++k4) {
                        const uint32_t koff = k4 * UMMA_K * 2;   // bytes
                        if (MODE == 0) {
                            const uint64_t a_hi = make_smem_desc(sbase + koff);
                            const uint64_t a_lo = make_smem_desc(sbase + A_BYTES + koff);
                            const uint64_t b_hi = make_smem_desc(sbase + 2 * A_BYTES + koff);
                            const uint64_t b_lo = make_smem_desc(sbase + 2 * A_BYTES + B_BYTES + koff);
                            umma_f16<kInstrDescBF16>(tmem_d, a_lo, b_hi, (kb | k4) != 0 ? 1u : 0u);   // small terms first
                            umma_f16<kInstrDescBF16>(tmem_d, a_hi, b_lo, 1u);
                            umma_f16<kInstrDescBF16>(tmem_d, a_hi, b_hi, 1u);
                        } else {
                            const uint64_t a_h = make_smem_desc(sbase + koff);
                            const uint64_t b_h = make_smem_desc(sbase + A_BYTES + koff);
                            umma_f16<kInstrDescF16>(tmem_d, a_h, b_h, (kb | k4) != 0 ? 1u : 0u);
                        }
                    }
                    umma_commit(empty_bar(stage));                       // frees the smem slot when the MMAs retire
                    if (kb == num_kb - 1) umma_commit(tfull_bar(buf));   // accumulator complete
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else {
        // ================================ epilogue ====================================
        const int quad = warp & 3;                 // TMEM lane quadrant this warp may access
        const int row = quad * 32 + lane;          // time bin inside the tile
        int it = 0;
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
            int ib, tb;
            decode_tile(g, tile, ib, tb);
            const int buf = it & 1;
            mbar_wait(tfull_bar(buf), (uint32_t)(it >> 1) & 1u);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(buf * BN);
            const int bin = ib * BM + row;
            // MODE 0: the stage-1 threshold itself.  MODE 1: thr1 lowered by the derived bound of the fp16 screen's
            // error for this (bin, template block), so that no true candidate can be missed (see file header).
            float thr_sq = g.thr1_sq;
            if (MODE == 1) {
                const float Bn = bin < g.M ? __ldg(g.bin_norm + bin) : 0.f;
                const float nmax = __ldg(g.tnorm_blk + tb);
                const float te = g.thr1 - (g.kappa1 * nmax * Bn + g.kappa2 * (Bn + nmax) + g.slack);
                thr_sq = te > 0.f ? te * te : 0.f;
            }
            epilogue_tile(g, taddr, bin, tb, lane, thr_sq);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(buf));
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS) : "memory");
    }
}


// ---------------------------------------------------------------------------------------------------------------
// Screen mode on CTA PAIRS (thread-block clusters of 2).  The two CTAs of a cluster work on the two halves of a
// 256-bin x 128-template super-tile: same coefficient tile (B operand, 32 KB per K block), different beta^avg rows
// (A operand).  Each CTA fetches only HALF of B and multicasts it into both CTAs' shared memory, so a CTA pulls
// 16 + 16 KB instead of 16 + 32 KB per K block from L2 -- the single-CTA kernel runs at 15 TB/s of L2 reads, which,
// not the MMA rate, is what limits it.  A stage may be refilled only when BOTH CTAs' MMAs have drained it: the
// tcgen05.commit that frees a stage arrives on the "empty" barrier of both CTAs (count 2).
namespace {

__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_id_x() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t num_clusters_x() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void tma_load_2d_mc(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y,
                                               uint16_t mask) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster"
        " [%0], [%1, {%3, %4}], [%2], %5;" ::"r"(dst),
        "l"(map), "r"(bar), "r"(x), "r"(y), "h"(mask)
        : "memory");
}
__device__ __forceinline__ void umma_commit_mc(uint32_t bar, uint16_t mask) {
    asm volatile(
        "tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(bar),
        "h"(mask)
        : "memory");
}

}  // namespace

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(NUM_THREADS, 1)
gemm_screen_pair_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmBh,
                        const GemmArgs g) {
    constexpr int STAGES = ModeCfg<1>::STAGES;
    constexpr uint32_t STAGE_BYTES = ModeCfg<1>::STAGE_BYTES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + b); };
    auto tempty_bar = [&](int b) { return bar_base + 8u * (2 * STAGES + 2 + b); };
    const uint32_t tmem_slot = bar_base + 8u * (2 * STAGES + 4);
    volatile uint32_t* tmem_slot_ptr =
        reinterpret_cast<volatile uint32_t*>(smem_raw + (tmem_slot - smem_u32(smem_raw)));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();

    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmBh) : "memory");
        for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 2); }
        for (int b = 0; b < 2; ++b) { mbar_init(tfull_bar(b), 1); mbar_init(tempty_bar(b), 4); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tmem_slot), "n"(TMEM_COLS)
                     : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();   // the peer's barriers are initialised before anything is multicast to them
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot_ptr;

    // super-tiles: pairs of time-bin blocks; both CTAs of a cluster walk the same sequence (lock step by construction)
    GemmArgs gp = g;
    gp.num_ib = (g.num_ib + 1) / 2;
    const int npairs = gp.num_tb * gp.num_ib;
    const int num_kb = (g.k2 + BK - 1) / BK;
    const int first = (int)cluster_id_x(), step = (int)num_clusters_x();

    if (warp == 0) {
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int pair = first; pair < npairs; pair += step) {
                int ibp, tb;
                decode_tile(gp, pair, ibp, tb);
                const int ib = 2 * ibp + (int)rank;   // may be one past the last block: TMA zero-fills, epilogue masks
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u);
                    const uint32_t sbase = smem_base + stage * STAGE_BYTES;
                    mbar_expect_tx(full_bar(stage), STAGE_BYTES);
                    tma_load_3d(sbase, &tmA, full_bar(stage), 0, ib * BM, kb);
                    // my half of the coefficient tile (128 of its 256 rows), into both CTAs
                    tma_load_2d_mc(sbase + A_BYTES + rank * (B_BYTES / 2), &tmBh, full_bar(stage), kb * BK,
                                   tb * BN + (int)rank * (BN / 2), (uint16_t)3);
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            int it = 0;
            for (int pair = first; pair < npairs; pair += step, ++it) {
                const int buf = it & 1;
                mbar_wait(tempty_bar(buf), ((uint32_t)(it >> 1) & 1u) ^ 1u);
                tc_fence_after();
                const uint32_t tmem_d = tmem_base + (uint32_t)(buf * BN);
                for (int kb = 0; kb < num_kb; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    const uint32_t sbase = smem_base + stage * STAGE_BYTES;
#pragma unroll
                    for (int k4 = 0; k4 < BK / UMMA_K; ++k4) {
                        const uint32_t koff = k4 * UMMA_K * 2;
                        const uint64_t a_h = make_smem_desc(sbase + koff);
                        const uint64_t b_h = make_smem_desc(sbase + A_BYTES + koff);
                        umma_f16<kInstrDescF16>(tmem_d, a_h, b_h, (kb | k4) != 0 ? 1u : 0u);
                    }
                    umma_commit_mc(empty_bar(stage), (uint16_t)3);       // frees the slot in BOTH CTAs
                    if (kb == num_kb - 1) umma_commit(tfull_bar(buf));
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else {
        const int quad = warp & 3;
        const int row = quad * 32 + lane;
        int it = 0;
        for (int pair = first; pair < npairs; pair += step, ++it) {
            int ibp, tb;
            decode_tile(gp, pair, ibp, tb);
            const int ib = 2 * ibp + (int)rank;
            const int buf = it & 1;
            mbar_wait(tfull_bar(buf), (uint32_t)(it >> 1) & 1u);
            tc_fence_after();
            const uint32_t taddr = tmem_base + ((uint32_t)(quad * 32) << 16) + (uint32_t)(buf * BN);
            const int bin = ib * BM + row;
            const float Bn = bin < g.M ? __ldg(g.bin_norm + bin) : 0.f;
            const float nmax = __ldg(g.tnorm_blk + tb);
            const float te = g.thr1 - (g.kappa1 * nmax * Bn + g.kappa2 * (Bn + nmax) + g.slack);
            const float thr_sq = te > 0.f ? te * te : 0.f;
            epilogue_tile(g, taddr, bin, tb, lane, thr_sq);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar(buf));
        }
    }

    tc_fence_before();
    __syncthreads();
    cluster_sync_all();   // no CTA retires while its peer may still multicast into it or arrive on its barriers
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(TMEM_COLS) : "memory");
    }
}

cudaError_t gemm_tcgen05_configure() {
    cudaError_t e = cudaFuncSetAttribute(gemm_tcgen05_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)ModeCfg<0>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(gemm_tcgen05_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)ModeCfg<1>::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(gemm_screen_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)ModeCfg<1>::SMEM_BYTES);
}

// How many 2-CTA clusters of the pair kernel the device can hold at once (0: use the single-CTA kernel).
cudaError_t gemm_screen_pair_clusters(int num_sms, int* clusters) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(num_sms / 2 * 2));
    cfg.blockDim = dim3(NUM_THREADS);
    cfg.dynamicSmemBytes = ModeCfg<1>::SMEM_BYTES;
    cudaLaunchAttribute attr;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = 2; attr.val.clusterDim.y = 1; attr.val.clusterDim.z = 1;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
    int n = 0;
    cudaError_t e = cudaOccupancyMaxActiveClusters(&n, gemm_screen_pair_kernel, &cfg);
    if (e != cudaSuccess) { cudaGetLastError(); n = 0; }
    *clusters = n;
    return cudaSuccess;
}

cudaError_t launch_gemm_tcgen05(const CUtensorMap& tmA_hi, const CUtensorMap& tmA_lo, const CUtensorMap& tmB_hi,
                                const CUtensorMap& tmB_lo, const GemmArgs& g, int num_sms, cudaStream_t st) {
    const int ntiles = g.num_tb * g.num_ib;
    const int grid = ntiles < num_sms ? ntiles : num_sms;
    gemm_tcgen05_kernel<0><<<grid, NUM_THREADS, ModeCfg<0>::SMEM_BYTES, st>>>(tmA_hi, tmA_lo, tmB_hi, tmB_lo, g);
    return cudaGetLastError();
}

cudaError_t launch_gemm_screen(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmB_half,
                               int pair_clusters, const GemmArgs& g, int num_sms, cudaStream_t st) {
    if (pair_clusters > 0) {
        const int npairs = g.num_tb * ((g.num_ib + 1) / 2);
        const int nc = npairs < pair_clusters ? npairs : pair_clusters;
        gemm_screen_pair_kernel<<<2 * nc, NUM_THREADS, ModeCfg<1>::SMEM_BYTES, st>>>(tmA, tmB_half, g);
        return cudaGetLastError();
    }
    const int ntiles = g.num_tb * g.num_ib;
    const int grid = ntiles < num_sms ? ntiles : num_sms;
    gemm_tcgen05_kernel<1><<<grid, NUM_THREADS, ModeCfg<1>::SMEM_BYTES, st>>>(tmA, tmA, tmB, tmB, g);
    return cudaGetLastError();
}

}  // namespace rbmf
