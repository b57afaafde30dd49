// Kernel 1 (steps a1-a3 of include/rbmf.h): pointwise correlation fused into a batched inverse FFT, the w-sample
// bin average fused into its last pass -- ONE persistent, warp-specialised launch whose intermediate stays in L2.
//
// Four-step FFT, N = L1 * L2, per basis column:
//   pass 1 (line = j2, length L1):  Y[n1][j2] = e^{2 pi i j2 n1 / N} sum_{j1} G[j1 L2 + j2] e^{2 pi i j1 n1 / L1}
//   pass 2 (line = n1, length L2):  beta[n1 + L1 n2] = sum_{j2} Y[n1][j2] e^{2 pi i j2 n2 / L2}
// with G[j] = s d[j] conj(b[j]) formed by pass 1 as it reads its inputs (a1) and zero for
// j >= N/2 (one-sided spectrum: the upper half of every pass-1 line is never read and its first radix-2 level is
// pruned).  beta^avg (a3, Eq. 9) sums w consecutive samples n = n1 + L1 n2, i.e. w consecutive lines
// n1 at equal n2: a pass-2 item owns max(w, SUB) consecutive lines and reduces their outputs through shared memory
// before writing the operand plane(s) of kernel 2.
//
// Columns are processed in chunks of C = 4 (32-byte row segments).  Work queue (global ticket counter):
//   P1(0) | P1(1) P2(0) | P1(2) P2(1) | ...   (pass 1 runs FftArgs::lookahead chunks ahead, see rbmf_api.cu) so
// chunk c's intermediate Y (N * 32 bytes) is written and read back while it is still in the 126 MB L2.  Y lives IN
// PLACE in the chunk's block of the beta array (Y[n1][j2] at the address of beta[n1 + L1 j2]): a pass-2 item reads
// exactly the addresses it then overwrites, so dirty Y lines are overwritten in L2 before they are evicted and only
// basis (read) and beta / planes (written) touch HBM.
//
// One CTA per SM, 16 consumer warps + a producer warpgroup of which one warp works:
//   warp 16      producer: draws tickets, waits for a chunk's pass-1 completion counter before its pass-2 items, and
//                moves every tile's input into one of three shared-memory tile buffers with bulk-async copies
//                (cp.async.bulk 1-D for the basis block and the strain slice of a pass-1 tile; a 3-D tensor map over
//                the beta array for the strided Y rows of a pass-2 tile), completion signalled on an mbarrier;
//   warps 0-7, 8-15  two consumer groups of 256 threads; tiles alternate strictly between them (tile i -> group
//                i & 1, buffer i % 3), so a group never waits on global-memory latency: its next tile is loaded while
//                it computes.  Groups synchronise internally with a named barrier (bar.sync id, 256).
// Inside a group a line of length L = R0 * R1 is two Stockham stages: a thread owns one column and R0 elements; stage 0
// reads its elements (positions wk + q W) from the tile buffer, does a radix-R0 DFT in registers and writes the results
// back IN PLACE (the same, thread-private positions); after the group barrier stage 1 reads R1 consecutive positions,
// applies the twiddles (table in shared memory) and does a radix-R1 DFT.  Pass 1 then multiplies by the inter-pass
// twiddle (product of two small tables) and stores Y straight to global memory; pass 2 writes its rows back to the tile
// buffer, where the bin sums read them, and one TMA tensor store moves them to the beta array.
// Tile buffer layout: [position][line][column] (one row = SUB lines x 4 columns), conflict-free for both stages; when
// a row is only 64 bytes (L = 1024) one pad row per 32 rows keeps stage 1 conflict-free.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "rbmf_internal.h"

namespace rbmf {

namespace {

constexpr int C = kFftC;
constexpr int GT = kFftThreads;         // threads per consumer group
constexpr int NGROUP = 2;
constexpr int NT = NGROUP * GT + 128;   // + producer warpgroup (one working warp; setmaxnreg acts on warpgroups)
constexpr int NBUF = 3;
constexpr int kE2Stride = GT / C + 2 * 16;   // per-group E2 factors: SUB lines of R1 entries, each line padded by 2

// ------------------------------------------------------------------------------------------------ complex helpers
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cmul_conj(float2 d, float2 b) {   // d * conj(b)
    return make_float2(d.x * b.x + d.y * b.y, d.y * b.x - d.x * b.y);
}
// Complex add / subtract as ONE packed fp32x2 instruction (FADD2 on sm_100): the butterflies are ~2/3 additions and
// the kernel is bound by instruction issue, not by the fp32 lanes.
__device__ __forceinline__ unsigned long long pk2(float2 a) {
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a.x), "f"(a.y));
    return r;
}
__device__ __forceinline__ float2 upk2(unsigned long long r) {
    float2 a;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(a.x), "=f"(a.y) : "l"(r));
    return a;
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a)), "l"(pk2(b)));
    return upk2(r);
}
__device__ __forceinline__ float2 csub(float2 a, float2 b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a)), "l"(pk2(b)));
    return upk2(r);
}

// v * e^{+2 pi i m / 32}, 0 <= m < 16; m is a compile-time constant after unrolling.
__device__ __forceinline__ float2 mul_w32(float2 v, int m) {
    constexpr float CS[9] = {1.0f,
                             0.98078528040323044913f,
                             0.92387953251128675613f,
                             0.83146961230254523708f,
                             0.70710678118654752440f,
                             0.55557023301960222474f,
                             0.38268343236508977173f,
                             0.19509032201612826785f,
                             0.0f};
    if (m == 0) return v;
    if (m == 8) return make_float2(-v.y, v.x);
    if (m == 4) return make_float2((v.x - v.y) * CS[4], (v.x + v.y) * CS[4]);
    if (m == 12) return make_float2((-v.x - v.y) * CS[4], (v.x - v.y) * CS[4]);
    const float c = m < 8 ? CS[m] : -CS[16 - m];
    const float s = m < 8 ? CS[8 - m] : CS[m - 8];
    return cmul(v, make_float2(c, s));
}

// In-register inverse DFT of length R (natural order in and out): x[m] <- sum_j x[j] e^{+2 pi i j m / R}.
template <int R>
__device__ __forceinline__ void dft(float2 (&x)[R]) {
    if constexpr (R == 2) {
        const float2 a = x[0], b = x[1];
        x[0] = cadd(a, b);
        x[1] = csub(a, b);
    } else {
        float2 e[R / 2], o[R / 2];
#pragma unroll
        for (int i = 0; i < R / 2; ++i) { e[i] = x[2 * i]; o[i] = x[2 * i + 1]; }
        dft<R / 2>(e);
        dft<R / 2>(o);
#pragma unroll
        for (int i = 0; i < R / 2; ++i) {
            const float2 t = mul_w32(o[i], i * (32 / R));
            x[i] = cadd(e[i], t);
            x[i + R / 2] = csub(e[i], t);
        }
    }
}

// Same, for an input whose upper half x[R/2 .. R) is zero (and not read): the deepest level degenerates to a copy.
template <int R>
__device__ __forceinline__ void dft_half(float2 (&x)[R]) {
    if constexpr (R == 2) {
        x[1] = x[0];
    } else {
        float2 e[R / 2], o[R / 2];
#pragma unroll
        for (int i = 0; i < R / 4; ++i) { e[i] = x[2 * i]; o[i] = x[2 * i + 1]; }
        dft_half<R / 2>(e);
        dft_half<R / 2>(o);
#pragma unroll
        for (int i = 0; i < R / 2; ++i) {
            const float2 t = mul_w32(o[i], i * (32 / R));
            x[i] = cadd(e[i], t);
            x[i + R / 2] = csub(e[i], t);
        }
    }
}

// ------------------------------------------------------------------------------------ mbarrier / bulk-copy helpers
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
// 1-D bulk copy global -> shared (16-byte aligned addresses, size a multiple of 16), completion on an mbarrier.
// L2 policies: the basis is streamed once (evict first); strain slice, Y and tables are re-read (evict last / normal).
__device__ __forceinline__ unsigned long long policy_evict_first() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ unsigned long long policy_evict_normal() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ unsigned long long policy_evict_last() {
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar,
                                         unsigned long long pol) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
        "l"(src), "r"(bytes), "r"(bar), "l"(pol)
        : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, uint32_t bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst),
        "l"(map), "r"(bar), "r"(x), "r"(y), "r"(z)
        : "memory");
}
// Tensor store shared -> global (bulk async group): the beta rows of a pass-2 tile leave through the same 3-D map
// their Y rows came in by.
// beta is written once and not read again by this kernel: evict-first keeps it from displacing the Y rows in L2.
__device__ __forceinline__ void tma_store_3d(const CUtensorMap* map, uint32_t src, int x, int y, int z) {
    const unsigned long long pol = policy_evict_first();
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3, %4}], [%1], %5;" ::"l"(map),
                 "r"(src), "r"(x), "r"(y), "r"(z), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void group_sync(int g) {   // named barrier of one consumer group
    if (g == 0) asm volatile("bar.sync 1, %0;" ::"n"(GT) : "memory");
    else asm volatile("bar.sync 2, %0;" ::"n"(GT) : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Poll with relaxed loads (an acquire load would invalidate the SM's L1 on every iteration).
__device__ __forceinline__ void wait_counter(const unsigned* p, unsigned target) {
    for (;;) {
        unsigned v;
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
        if (v >= target) break;
        __nanosleep(100);
    }
    __threadfence();
    asm volatile("fence.proxy.async;" ::: "memory");   // the guarded data is read next through the async proxy (TMA)
}

// ------------------------------------------------------------------------------------------- per-length config
// PASS1: the pass-1 tile buffer may carry pad rows (its producer uses 1-D bulk copies, 16-byte aligned); pass-2 tiles
// arrive through tensor copies whose destination must stay 128-byte aligned, so they are never padded.
template <int LOGL, bool PASS1>
struct Cfg {
    static constexpr int L = 1 << LOGL;
    static constexpr int R0 = fft_r0(LOGL);
    static constexpr int R1 = fft_r1(LOGL);
    static constexpr int W = R1;                      // threads per column per line
    static constexpr int SUB = GT / (R1 * C);         // lines per tile
    static constexpr int RB = SUB * C;                // float2 per tile-buffer row (one position: SUB lines x C columns)
    static constexpr bool PAD = PASS1 && RB * 8 == 64;   // 64-byte rows: one pad row per 32 rows
    static constexpr int ROWS = PAD ? L + L / 32 : L;
    static constexpr int TILE_F2 = ROWS * RB;         // float2 per tile buffer
    // strain slice of a pass-1 tile: one row of H values per line, rows offset so that the SUB lines a warp reads at
    // once fall into different banks
    static constexpr int SPAD = fft_spad(LOGL);
    __device__ static __forceinline__ int idx(int p) { return PAD ? p + (p >> 5) : p; }
};

enum TileType : int { TILE_NOP = 0, TILE_P1 = 1, TILE_P2 = 2, TILE_STOP = 3 };

// Cycle accounting of the producer / consumer hand-off (build with -DRBMF_FFT_PROFILE; read by rbmf_fft_profile_read).
#ifdef RBMF_FFT_PROFILE
__device__ unsigned long long g_fft_prof[32];
#define PROF_T() clock64()
#define PROF_ADD(i, v) atomicAdd(&g_fft_prof[i], (unsigned long long)(v))
#else
#define PROF_T() 0ll
#define PROF_ADD(i, v) ((void)0)
#endif

template <int LOG1, int LOG2>
struct Smem {
    static constexpr int BUF_F2 = Cfg<LOG1, true>::TILE_F2 > Cfg<LOG2, false>::TILE_F2 ? Cfg<LOG1, true>::TILE_F2
                                                                                         : Cfg<LOG2, false>::TILE_F2;
    static constexpr size_t BUF_BYTES = (size_t)BUF_F2 * 8;
    static constexpr size_t TW_A = NBUF * BUF_BYTES;                      // tw1_a: L1 float2
    static constexpr size_t TW_B = TW_A + ((size_t)8 << LOG1);            // tw1_b: L2 float2
    static constexpr size_t BARS = TW_B + ((size_t)8 << LOG2);            // full[NBUF][NGROUP], empty[NBUF]
    static constexpr size_t E2S = BARS + 3 * NBUF * 8;                    // float2 e2s[NGROUP][kE2Stride]
    static constexpr size_t META = E2S + NGROUP * kE2Stride * 8;          // int4 meta[2 NBUF]: tile descriptors (ring)
    static constexpr size_t TOTAL = META + 2 * NBUF * 16 + 128 /* base alignment slack */;
};

// ------------------------------------------------------------------------------------------- pass 1 (consumer)
// Tile = SUB consecutive lines j2 of one chunk.  Thread (col, line, wk) of the group.  On entry rows [0, H) of the tile
// buffer hold the basis block [j1][line][col] and rows [H, ...) the strain slice [line][j1] (both placed by the
// producer); stage 0 multiplies them (a1), transforms along j1 and writes back in place.
template <int LOG1, int LOG2>
__device__ __forceinline__ void p1_tile(const FftArgs& a, int g, int gt, int chunk, int tile, float2* B,
                                        const float2* tw1, float2* e2s) {
    using K = Cfg<LOG1, true>;
    constexpr int L1 = K::L, R0 = K::R0, R1 = K::R1, W = K::W, H = L1 / 2, SUB = K::SUB, RB = K::RB;
    const int col = gt % C, line = (gt / C) % SUB, wk = gt / (C * SUB);
    const int slot = line * C + col;
    const int j2 = tile * SUB + line;

    // Inter-pass twiddle e^{2 pi i j2 n1 / N}, n1 = b + m R0, as the product E1[j2][b] E2[j2][m]: this thread's E1
    // factors are fetched now and used in stage 1; the SUB x R1 = 64 E2 factors of the tile go to shared memory.
    constexpr int NB = R0 / R1, L2 = 1 << LOG2;
    float2 e1[NB];
#pragma unroll
    for (int bb = 0; bb < NB; ++bb) e1[bb] = __ldg(a.twN + (size_t)j2 * R0 + wk + bb * W);
    // (lines are padded by two entries: the lanes of a warp read the same entry of 2+ different lines at once)
    if (gt < SUB * R1) e2s[gt + 2 * (gt / R1)] = __ldg(a.twN + (size_t)L2 * R0 + (size_t)(tile * SUB) * R1 + gt);

    // ---- a1 + stage 0 ---------------------------------------------------------------------------------
    float2 u[R0];
    {
        const float2* S = B + K::idx(H) * RB + line * (H + K::SPAD);
#pragma unroll
        for (int q = 0; q < R0 / 2; ++q) {
            const int j1 = wk + q * W;
            u[q] = cmul_conj(S[j1], B[K::idx(j1) * RB + slot]);
        }
    }
    group_sync(g);   // the strain slice sits where stage 0 writes its upper-half results
    dft_half<R0>(u);
#pragma unroll
    for (int m = 0; m < R0; ++m) B[K::idx(wk + m * W) * RB + slot] = u[m];
    group_sync(g);

    // ---- stage 1 + inter-pass twiddle + store of Y (in place in the beta array) -------------------------------
    // virtual chunk = c * nb + b: basis chunk c against segment b's strain; beta arrays are [segment][chunk]
    const int bc = a.seg_major ? chunk % a.nchunk : chunk / a.nb, bs = a.seg_major ? chunk / a.nchunk : chunk % a.nb;
    float2* yrow = a.beta + ((size_t)(bs * a.nchunk + bc) * (size_t)a.N + (size_t)j2 * L1) * C + col;
    const float2* e2 = e2s + line * (R1 + 2);
#pragma unroll
    for (int bb = 0; bb < NB; ++bb) {
        const int b = wk + bb * W;   // butterfly index < R0
        float2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) x[q] = B[K::idx(b * R1 + q) * RB + slot];
#pragma unroll
        for (int q = 1; q < R1; ++q) x[q] = cmul(x[q], tw1[q * R0 + b]);
        dft<R1>(x);
#pragma unroll
        for (int m = 0; m < R1; ++m) {
            const int n1 = b + m * R0;
            __stcg(yrow + n1 * C, cmul(cmul(x[m], e2[m]), e1[bb]));
        }
    }
}

// ------------------------------------------------------------------------------------------- pass 2 (consumer)
__device__ __forceinline__ void store_plane_fp16(uint16_t* p, float2 v) {
    *reinterpret_cast<__half2*>(p) = __floats2half2_rn(v.x, v.y);
}
__device__ __forceinline__ void store_planes_bf16(uint16_t* phi, uint16_t* plo, float2 v) {
    const __nv_bfloat16 hx = __float2bfloat16_rn(v.x), hy = __float2bfloat16_rn(v.y);
    const __nv_bfloat16 lx = __float2bfloat16_rn(v.x - __bfloat162float(hx));
    const __nv_bfloat16 ly = __float2bfloat16_rn(v.y - __bfloat162float(hy));
    *reinterpret_cast<ushort2*>(phi) = make_ushort2(__bfloat16_as_ushort(hx), __bfloat16_as_ushort(hy));
    *reinterpret_cast<ushort2*>(plo) = make_ushort2(__bfloat16_as_ushort(lx), __bfloat16_as_ushort(ly));
}
__device__ __forceinline__ void store_planes(const FftArgs& a, int bin, int gcol, float2 v) {
    const size_t e = ((size_t)(gcol / 32) * a.M + bin) * 64 + (gcol % 32) * 2;
    if (a.plane_fp16) {
        // screen mode: one fp16 plane (round to nearest; |v| > 65504 becomes inf, which the screen lets through)
        *reinterpret_cast<__half2*>(a.plane_hi + e) = __floats2half2_rn(v.x, v.y);
        return;
    }
    const __nv_bfloat16 hx = __float2bfloat16_rn(v.x), hy = __float2bfloat16_rn(v.y);
    const __nv_bfloat16 lx = __float2bfloat16_rn(v.x - __bfloat162float(hx));
    const __nv_bfloat16 ly = __float2bfloat16_rn(v.y - __bfloat162float(hy));
    *reinterpret_cast<ushort2*>(a.plane_hi + e) = make_ushort2(__bfloat16_as_ushort(hx), __bfloat16_as_ushort(hy));
    *reinterpret_cast<ushort2*>(a.plane_lo + e) = make_ushort2(__bfloat16_as_ushort(lx), __bfloat16_as_ushort(ly));
}

// One round = SUB consecutive lines n1 = n1_r .. of one chunk (an item of span = max(w, SUB) lines is `rounds`
// consecutive rounds of the same group; acc carries the bin sums across them).  On entry the tile buffer holds the Y
// rows [j2][line][col].
template <int LOG1, int LOG2, int NIT>
__device__ __forceinline__ void p2_round(const FftArgs& a, const CUtensorMap* tmY, int g, int gt, int chunk, int n1_0,
                                         int rd, int rounds, float2* B, const float2* tw1, float2 (&acc)[NIT]) {
    using K = Cfg<LOG2, false>;
    constexpr int L1 = 1 << LOG1, L2 = K::L, R0 = K::R0, R1 = K::R1, W = K::W, SUB = K::SUB, RB = K::RB;
    const int col = gt % C, line = (gt / C) % SUB, wk = gt / (C * SUB);
    const int slot = line * C + col;
    const int w = a.w;
    const int bc = a.seg_major ? chunk % a.nchunk : chunk / a.nb, bs = a.seg_major ? chunk / a.nchunk : chunk % a.nb;
    const int zc = bs * a.nchunk + bc;                     // the chunk's block of the beta array
    const int gcol = bc * C + col;
    const int bin0 = bs * a.Mseg;                          // the segment's first row of the planes

    float2 u[R0];
#pragma unroll
    for (int q = 0; q < R0; ++q) u[q] = B[K::idx(wk + q * W) * RB + slot];
    dft<R0>(u);
#pragma unroll
    for (int m = 0; m < R0; ++m) B[K::idx(wk + m * W) * RB + slot] = u[m];
    group_sync(g);
#pragma unroll
    for (int bb = 0; bb < R0 / R1; ++bb) {
        const int b = wk + bb * W;
        float2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) x[q] = B[K::idx(b * R1 + q) * RB + slot];
#pragma unroll
        for (int q = 1; q < R1; ++q) x[q] = cmul(x[q], tw1[q * R0 + b]);
        dft<R1>(x);
#pragma unroll
        for (int m = 0; m < R1; ++m) {
            u[bb * R1 + m] = x[m];   // output n2 = b + m R0
        }
    }
    // ---- a3: sum the outputs of min(w, SUB) consecutive lines at equal n2 ----------------------------------------
    group_sync(g);   // every stage-1 read of the tile buffer is done
#pragma unroll
    for (int bb = 0; bb < R0 / R1; ++bb)
#pragma unroll
        for (int m = 0; m < R1; ++m) B[K::idx((wk + bb * W) + m * R0) * RB + slot] = u[bb * R1 + m];
    // The buffer now holds the tile's beta rows [n2][line][col] -- the layout of the beta array itself (in place of the
    // Y rows this tile loaded): one thread hands them to the TMA, the bin sums below read the same rows meanwhile.
    fence_async_smem();
    group_sync(g);
    if (gt == 0) {
        constexpr int BR = L2 < 256 ? L2 : 256;
        const int x = (n1_0 + rd * SUB) * C * 2;
        for (int p = 0; p < L2 / BR; ++p) tma_store_3d(tmY, smem_u32(B + (size_t)p * BR * RB), x, p * BR, zc);
        bulk_commit();
    }
    if (rd == 0) {
#pragma unroll
        for (int it = 0; it < NIT; ++it) acc[it] = make_float2(0.f, 0.f);
    }
    if (a.no_planes) {
        // template routes (template_route.cu): the caller reads beta itself; no operand planes for kernel 2
    } else if (w >= SUB) {
        // all SUB lines of this round fall into one bin per n2; a bin spans `rounds` rounds.  Each thread starts at
        // a different line (rot) so that the 16 lanes of a shared-memory wavefront hit 16 distinct 8-byte banks.
        const int rot = (gt >> (RB * 8 == 64 ? 3 : 2)) & (SUB - 1);
#pragma unroll
        for (int it = 0; it < NIT; ++it) {
            const int e = gt + it * GT;   // (n2, col): col is this thread's own
            if (L2 * C >= GT || e < L2 * C) {
                const int n2 = e / C;
                const float2* row = B + K::idx(n2) * RB + col;
                float2 sum = row[rot * C];
#pragma unroll
                for (int rr = 1; rr < SUB; ++rr) sum = cadd(sum, row[((rot + rr) & (SUB - 1)) * C]);
                acc[it] = cadd(acc[it], sum);
            }
        }
        if (rd == rounds - 1) {
            // bins n1_0 / w + (L1 / w) n2, n2 = gt / C + it GT / C: a constant element stride between iterations
            const size_t e0 = ((size_t)(gcol / 32) * a.M + bin0 + n1_0 / w + (size_t)(L1 / w) * (gt / C)) * 64 + (gcol % 32) * 2;
            const size_t es = (size_t)(L1 / w) * (GT / C) * 64;
            const float iw = a.inv_w;
            if (a.plane_fp16) {
#pragma unroll
                for (int it = 0; it < NIT; ++it)
                    if (L2 * C >= GT || gt + it * GT < L2 * C)
                        store_plane_fp16(a.plane_hi + e0 + it * es, make_float2(acc[it].x * iw, acc[it].y * iw));
            } else {
#pragma unroll
                for (int it = 0; it < NIT; ++it)
                    if (L2 * C >= GT || gt + it * GT < L2 * C)
                        store_planes_bf16(a.plane_hi + e0 + it * es, a.plane_lo + e0 + it * es,
                                          make_float2(acc[it].x * iw, acc[it].y * iw));
            }
        }
    } else {
        // w < SUB (including w = 1): this round completes SUB / w bins per n2; compact, not unrolled
        const int nb = SUB / w;
#pragma unroll 1
        for (int e = gt; e < nb * L2 * C; e += GT) {
            const int rb = e / (L2 * C), n2 = (e % (L2 * C)) / C;
            const float2* row = B + K::idx(n2) * RB + col;
            float2 sum = row[(rb * w) * C];
#pragma unroll 1
            for (int rr = 1; rr < w; ++rr) sum = cadd(sum, row[(rb * w + rr) * C]);
            store_planes(a, bin0 + (n1_0 + rd * SUB + rb * w) / w + (L1 / w) * n2, gcol,
                         make_float2(sum.x * a.inv_w, sum.y * a.inv_w));
        }
    }
    if (gt == 0) bulk_wait_read();   // the tensor store has read the buffer: it may be handed back to the producer
}

// ------------------------------------------------------------------------------------------------------ kernel
template <int LOG1, int LOG2>
__global__ void __launch_bounds__(NT, 1) fft_tma_kernel(const __grid_constant__ CUtensorMap tmY, const FftArgs a) {
    using K1 = Cfg<LOG1, true>;
    using K2 = Cfg<LOG2, false>;
    using S = Smem<LOG1, LOG2>;
    constexpr int L1 = 1 << LOG1, L2 = 1 << LOG2, H = L1 / 2;
    constexpr int NIT = (L2 * C + GT - 1) / GT;   // reduced outputs per thread and round
    extern __shared__ uint8_t smem_raw[];
    // 128-byte aligned base, derived by pointer arithmetic so that the compiler keeps the shared address space
    // (LDS / STS instead of generic loads and stores)
    uint8_t* sm = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    float2* tw_a = reinterpret_cast<float2*>(sm + S::TW_A);
    float2* tw_b = reinterpret_cast<float2*>(sm + S::TW_B);
    const uint32_t bars = smem_u32(sm + S::BARS);
    // One "full" barrier per (buffer, group): a parity wait can only tell the current phase from the previous one, and
    // a group that got an empty (NOP) tile may ask for its next tile in buffer b before the OTHER group's tile in b
    // has even landed -- on a barrier shared by both groups that request would alias to an older phase and pass.
    // With per-group barriers a group's successive waits on one barrier are successive phases (tiles i, i + 6, ...).
    auto full_bar = [&](int b, int g) { return bars + 8u * (b * NGROUP + g); };
    auto empty_bar = [&](int b) { return bars + 8u * (NBUF * NGROUP + b); };
    volatile int4* meta = reinterpret_cast<volatile int4*>(sm + S::META);
    float2* e2s_all = reinterpret_cast<float2*>(sm + S::E2S);
    auto buf_ptr = [&](int b) { return reinterpret_cast<float2*>(sm + (size_t)b * S::BUF_BYTES); };

    const int n1t = L2 / K1::SUB;                                  // pass-1 tiles per chunk
    const int span = a.w > K2::SUB ? a.w : K2::SUB;
    const int rounds = span / K2::SUB;
    const int n2t = L1 / span;                                     // pass-2 items per chunk
    const int per = n1t + n2t;
    const int nvc = a.nchunk * a.nb;                               // virtual chunks (basis chunk, segment)
    const int total = nvc * per;

    for (int i = threadIdx.x; i < L1; i += NT) tw_a[i] = a.tw1_a[i];
    for (int i = threadIdx.x; i < L2; i += NT) tw_b[i] = a.tw1_b[i];
    if (threadIdx.x == 0) {
        for (int b = 0; b < NBUF; ++b) {
            mbar_init(full_bar(b, 0), 1); mbar_init(full_bar(b, 1), 1); mbar_init(empty_bar(b), 1);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        fence_async_smem();
    }
    __syncthreads();

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp >= NGROUP * (GT / 32)) {
        // the producer needs few registers: hand the rest of the register file to the consumer warpgroups
        asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
        if (warp > NGROUP * (GT / 32)) return;
        // =========================================== producer ===========================================
        if (lane == 0) asm volatile("prefetch.tensormap [%0];" ::"l"(&tmY) : "memory");
        const unsigned long long pol_first = policy_evict_first(), pol_last = policy_evict_last(),
                                 pol_normal = policy_evict_normal();
        int next_ticket = 0;
        if (lane == 0) next_ticket = (int)atomicAdd(a.sched, 1u);
        // open pass-2 items of the two groups, as scalars (an array indexed by the group would live in local memory)
        int oc0 = 0, on0 = 0, or0 = 0, oc1 = 0, on1 = 0, or1 = 0;
        bool open0 = false, open1 = false;
        // n1t and n2t are powers of two; the one true division of the ticket decode, by per = n1t + n2t, is done with
        // a float reciprocal and a correction (tickets stay below 2^24, where float holds them exactly)
        const int lg_n1t = 31 - __clz(n1t), lg_n2t = 31 - __clz(n2t);
        const float inv_per = 1.0f / (float)per;
        const int la = nvc < a.lookahead ? nvc : a.lookahead, nfull = nvc - la;
        int stops = 0;
        for (int i = 0; stops < NGROUP; ++i) {
            const int g = i & 1, buf = i % NBUF;
            const uint32_t use = (uint32_t)(i / NBUF);
            int type = TILE_NOP, chunk = 0, idx = 0, rd = 0;
            [[maybe_unused]] const long long pt0 = PROF_T();
            [[maybe_unused]] long long pt_dep = 0, pt1 = 0, pt2 = 0;
            if (lane == 0) {
                // The tile is chosen (ticket decoded, a pass-2 item's dependency on its chunk's pass-1 counter waited
                // for) BEFORE the wait for the buffer: that latency then overlaps the consumers' work on the buffer.
                const bool my_open = g ? open1 : open0, other_open = g ? open0 : open1;
                if (my_open) {
                    type = TILE_P2; chunk = g ? oc1 : oc0; idx = g ? on1 : on0; rd = g ? or1 : or0;
                } else if (next_ticket < total) {
                    const int t = next_ticket;
                    next_ticket = (int)atomicAdd(a.sched, 1u);
                    // queue order, pass 1 running LA chunks ahead of pass 2:
                    //   P1(0) .. P1(LA-1) | P1(LA) P2(0) | P1(LA+1) P2(1) | ... | P2(n-LA) | ... | P2(n-1)
                    bool first = true;
                    if (t < (la << lg_n1t)) {
                        chunk = t >> lg_n1t; idx = t & (n1t - 1);
                    } else {
                        const int u = t - (la << lg_n1t);
                        if (u < nfull * per) {
                            int blk = (int)((float)u * inv_per);
                            if (blk * per > u) --blk;
                            else if ((blk + 1) * per <= u) ++blk;
                            const int v = u - blk * per;
                            if (v < n1t) { chunk = blk + la; idx = v; }
                            else { first = false; chunk = blk; idx = v - n1t; }
                        } else {
                            const int u2 = u - nfull * per;
                            first = false; chunk = nfull + (u2 >> lg_n2t); idx = u2 & (n2t - 1);
                        }
                    }
                    if (first) {
                        type = TILE_P1;
                    } else {
                        type = TILE_P2; idx *= span; rd = 0;
                        [[maybe_unused]] const long long d0 = PROF_T();
                        wait_counter(a.sched + kSchedBase + chunk, (unsigned)n1t);   // all of the chunk's Y is in L2
                        pt_dep = PROF_T() - d0;
                    }
                } else if (!other_open) {
                    type = TILE_STOP;
                }
                // Everything the copies need is worked out, and the tile's descriptor published (the meta ring has
                // 2 NBUF slots, so the slot of the tile still being processed in this buffer is not touched), BEFORE the
                // wait for the buffer: once the consumers release it only expect_tx + the copies remain on the path.
                const int ms = i % (2 * NBUF);
                meta[ms].x = type; meta[ms].y = chunk; meta[ms].z = idx; meta[ms].w = rd;
                const uint32_t dst = smem_u32(buf_ptr(buf));
                // virtual chunk = c * nb + b (chunk-major: a basis chunk serves all segments from L2) or b * nchunk + c
                const int bc = a.seg_major ? chunk % a.nchunk : chunk / a.nb, bs = a.seg_major ? chunk / a.nchunk : chunk % a.nb;
                // both parts of a pass-1 tile sit in global memory in tile-buffer order (rbmf_internal.h): one bulk copy each
                constexpr uint32_t basis_bytes = (uint32_t)fft_p1_rows(LOG1) * K1::RB * 8;
                constexpr uint32_t strain_bytes = (uint32_t)K1::SUB * fft_strain_row(LOG1) * 8;
                static_assert(fft_p1_rows(LOG1) == (K1::PAD ? H + H / 32 : H) && fft_strain_row(LOG1) == H + K1::SPAD, "tile layout");
                static_assert(basis_bytes % 16 == 0 && strain_bytes % 16 == 0, "bulk copies move multiples of 16 bytes");
                const float2* src_basis = a.basisP + ((size_t)bc * n1t + idx) * (size_t)(fft_p1_rows(LOG1) * K1::RB);
                const float2* src_strain = a.dsT + ((size_t)bs * L2 + (size_t)idx * K1::SUB) * fft_strain_row(LOG1);
                // a basis chunk is streamed from HBM once per call: later segments of a batch find it in L2
                const unsigned long long pol_basis = (a.seg_major || bs == a.nb - 1) ? pol_first : pol_normal;
                constexpr int BR = L2 < 256 ? L2 : 256;          // rows per tensor copy of a pass-2 tile
                const int x = (idx + rd * K2::SUB) * C * 2;      // floats along the (n1, col) axis
                const int zc = bs * a.nchunk + bc;               // the chunk's block of the beta array
                const uint32_t fb = full_bar(buf, g);
                pt1 = PROF_T();
                mbar_wait(empty_bar(buf), (use & 1u) ^ 1u);
                pt2 = PROF_T();
                if (type == TILE_P1) {
                    mbar_expect_tx(fb, basis_bytes + strain_bytes);
                    bulk_g2s(dst, src_basis, basis_bytes, fb, pol_basis);
                    bulk_g2s(dst + basis_bytes, src_strain, strain_bytes, fb, pol_last);
                } else if (type == TILE_P2) {
                    mbar_expect_tx(fb, (uint32_t)L2 * K2::RB * 8);
#pragma unroll
                    for (int p = 0; p < L2 / BR; ++p)
                        tma_load_3d(dst + (uint32_t)K2::idx(p * BR) * K2::RB * 8, &tmY, fb, x, p * BR, zc);
                    const bool more = rd + 1 < rounds;
                    if (g) { open1 = more; oc1 = chunk; on1 = idx; or1 = rd + 1; }
                    else { open0 = more; oc0 = chunk; on0 = idx; or0 = rd + 1; }
                } else {
                    mbar_arrive(fb);
                }
            }
            if (__shfl_sync(0xffffffffu, type, 0) == TILE_STOP) ++stops;
            __syncwarp();
            if (lane == 0) {
                PROF_ADD(0, 1); PROF_ADD(1, pt1 - pt0 - pt_dep); PROF_ADD(2, pt_dep); PROF_ADD(3, pt2 - pt1);
                PROF_ADD(4, PROF_T() - pt2);
            }
        }
    } else {
        // =========================================== consumers ==========================================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 112;");
        const int g = warp / (GT / 32), gt = threadIdx.x - g * GT;
        float2 acc[NIT];
#pragma unroll
        for (int it = 0; it < NIT; ++it) acc[it] = make_float2(0.f, 0.f);
        for (int i = g;; i += NGROUP) {
            const int buf = i % NBUF;
            [[maybe_unused]] const long long ct0 = PROF_T();
            mbar_wait(full_bar(buf, g), (uint32_t)(i / (NBUF * NGROUP)) & 1u);
            [[maybe_unused]] const long long ct1 = PROF_T();
            const int ms = i % (2 * NBUF);
            const int type = meta[ms].x, chunk = meta[ms].y, idx = meta[ms].z, rd = meta[ms].w;
            if (type == TILE_STOP) break;
            float2* B = buf_ptr(buf);
            if (type == TILE_P1) p1_tile<LOG1, LOG2>(a, g, gt, chunk, idx, B, tw_a, e2s_all + g * kE2Stride);
            else if (type == TILE_P2) p2_round<LOG1, LOG2, NIT>(a, &tmY, g, gt, chunk, idx, rd, rounds, B, tw_b, acc);
            fence_async_smem();   // this thread's generic-proxy writes to the buffer, before the async proxy refills it
            group_sync(g);
            if (gt == 0) {
                PROF_ADD(8 + 4 * type, 1); PROF_ADD(9 + 4 * type, ct1 - ct0); PROF_ADD(10 + 4 * type, PROF_T() - ct1);
                mbar_arrive(empty_bar(buf));
                if (type == TILE_P1) {
                    // release: the group's Y stores happen before this fence through the barrier above (bar.sync
                    // orders them at CTA scope, the gpu-scope fence is cumulative), then the counter is bumped
                    __threadfence();
                    atomicAdd(a.sched + kSchedBase + chunk, 1u);
                }
            }
        }
        if (gt == 0) bulk_wait_all();   // this thread's beta stores are complete before the CTA retires
    }
}

template <int LOG1, int LOG2>
cudaError_t configure_one(size_t* smem_bytes) {
    constexpr size_t smem = Smem<LOG1, LOG2>::TOTAL;
    *smem_bytes = smem;
    return cudaFuncSetAttribute(fft_tma_kernel<LOG1, LOG2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

template <int LOG1, int LOG2>
cudaError_t launch_one(const CUtensorMap& tmY, const FftArgs& a, int grid, cudaStream_t st) {
    fft_tma_kernel<LOG1, LOG2><<<grid, NT, Smem<LOG1, LOG2>::TOTAL, st>>>(tmY, a);
    return cudaGetLastError();
}

}  // namespace

// N = 2^(logL1 + logL2) with logL1 = ceil(n/2), logL2 = floor(n/2), n = 10 .. 20.
#define RBMF_FFT_DISPATCH(FN, ...)                                   \
    switch (logL1 * 16 + logL2) {                                    \
        case 5 * 16 + 5: return FN<5, 5>(__VA_ARGS__);               \
        case 6 * 16 + 5: return FN<6, 5>(__VA_ARGS__);               \
        case 6 * 16 + 6: return FN<6, 6>(__VA_ARGS__);               \
        case 7 * 16 + 6: return FN<7, 6>(__VA_ARGS__);               \
        case 7 * 16 + 7: return FN<7, 7>(__VA_ARGS__);               \
        case 8 * 16 + 7: return FN<8, 7>(__VA_ARGS__);               \
        case 8 * 16 + 8: return FN<8, 8>(__VA_ARGS__);               \
        case 9 * 16 + 8: return FN<9, 8>(__VA_ARGS__);               \
        case 9 * 16 + 9: return FN<9, 9>(__VA_ARGS__);               \
        case 10 * 16 + 9: return FN<10, 9>(__VA_ARGS__);             \
        case 10 * 16 + 10: return FN<10, 10>(__VA_ARGS__);           \
        default: return cudaErrorInvalidValue;                       \
    }

#ifdef RBMF_FFT_PROFILE
extern "C" int rbmf_fft_profile_read(unsigned long long* out32, int reset) {
    cudaDeviceSynchronize();
    if (cudaMemcpyFromSymbol(out32, g_fft_prof, sizeof(g_fft_prof)) != cudaSuccess) return -1;
    if (reset) {
        unsigned long long z[32] = {};
        if (cudaMemcpyToSymbol(g_fft_prof, z, sizeof(z)) != cudaSuccess) return -1;
    }
    return 0;
}
#endif

cudaError_t fft_tma_configure(int logL1, int logL2, size_t* smem_bytes) {
    RBMF_FFT_DISPATCH(configure_one, smem_bytes)
}

cudaError_t launch_fft_tma(const CUtensorMap& tmY, const FftArgs& a, int logL1, int logL2, int grid, cudaStream_t st) {
    RBMF_FFT_DISPATCH(launch_one, tmY, a, grid, st)
}


}  // namespace rbmf
