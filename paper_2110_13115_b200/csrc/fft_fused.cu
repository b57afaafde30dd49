// Kernel 1 (steps a1-a3 of include/rbmf.h): pointwise correlation fused into a batched inverse FFT, the w-sample
// bin average fused into its last pass, all in ONE persistent launch whose intermediate stays in L2.
//
// Four-step FFT, N = L1 * L2, per basis column:
//   pass 1 (line = j2, length L1):  Y[n1][j2] = e^{2 pi i j2 n1 / N} sum_{j1} G[j1 L2 + j2] e^{2 pi i j1 n1 / L1}
//   pass 2 (line = n1, length L2):  beta[n1 + L1 n2] = sum_{j2} Y[n1][j2] e^{2 pi i j2 n2 / L2}
// with G[j] = s d[j] conj(b[j]) formed in registers by pass 1's loads (a1) and zero for
// j >= N/2 (one-sided spectrum: the upper half of every pass-1 line is never read and its first radix-2 level is
// pruned).  beta^avg (a3, Eq. 9) is the sum of w consecutive samples n = n1 + L1 n2, i.e. of w
// consecutive lines n1 at equal n2: a pass-2 work item owns max(w, SUB) consecutive lines and reduces their
// outputs through shared memory before writing the bf16 hi/lo operand planes of kernel 2.
//
// Columns are processed in chunks of C = 4 (32-byte row segments).  The work queue is ordered
//   P1(0) P1(1) P2(0) P1(2) P2(1) ... so that chunk c's intermediate Y (N * 32 bytes) is written and read back while
// it is still in the 126 MB L2.  Y lives IN PLACE in the chunk's block of the beta array (Y[n1][j2] at the address
// of beta[n1 + L1 j2]): a pass-2 item reads exactly the addresses it then overwrites, dirty Y lines are normally
// overwritten in L2 before they are ever evicted, and only the basis (read) and beta / planes (written) touch HBM.
// CTAs draw tickets from a global counter; a pass-2 item waits on its chunk's pass-1 completion counter.  Every
// waited-on ticket is lower than the waiting one and already owned by a running CTA, so the scheme cannot deadlock.
//
// Inside a CTA (256 threads) a line of length L = R0 * R1 is two Stockham stages: a thread owns one column and R0
// elements, computes a radix-R0 butterfly in registers, exchanges through padded shared memory, then R0/R1
// butterflies of radix R1.  SUB = 256 / (R1 * C) lines are processed in lockstep.  All layouts (basis, Y, beta,
// planes) are chosen so that the 32 lanes of a warp always touch 128..256 contiguous bytes.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "rbmf_internal.h"

namespace rbmf {

namespace {

constexpr int C = kFftC;
constexpr int NT = kFftThreads;

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cmul_conj(float2 d, float2 b) {   // d * conj(b)
    return make_float2(d.x * b.x + d.y * b.y, d.y * b.x - d.x * b.y);
}
// Complex add / subtract as ONE packed fp32x2 instruction (FADD2 on sm_100): the butterflies are ~2/3 additions, and
// the kernel is bound by instruction issue, not by the fp32 lanes (a packed op does two lanes' work per issue slot).
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
    // cos(2 pi m / 32), sin(2 pi m / 32) from the first-octant table
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

// Streaming loads / stores: the basis is read once (no L1 allocation), Y lives in L2 only (never in the
// non-coherent L1: ring slots are rewritten by other SMs), beta and the planes are written once.
__device__ __forceinline__ float2 ld_stream(const float2* p) {
    float2 v;
    asm volatile("ld.global.nc.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// Poll with relaxed loads (an acquire load would invalidate the SM's L1 on every iteration); the data guarded by
// the counter (Y) is read with ld.global.cg, i.e. from L2, the point of coherence, after the CTA barrier that
// follows this wait.
__device__ __forceinline__ void wait_counter(const unsigned* p, unsigned target) {
    for (;;) {
        unsigned v;
        asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
        if (v >= target) break;
        __nanosleep(100);
    }
    __threadfence();
}

template <int LOGL>
struct Cfg {
    static constexpr int L = 1 << LOGL;
    static constexpr int R0 = fft_r0(LOGL);
    static constexpr int R1 = fft_r1(LOGL);
    static constexpr int W = R1;                   // threads per column per line
    static constexpr int SUB = fft_sub(LOGL);      // lines per CTA in lockstep
    static constexpr int ROWS = R1 * (R0 + 1);     // padded exchange rows per line (>= L)
    // lines touched by one warp: pass 1 maps tid -> (col, wk, line), pass 2 maps tid -> (col, line, wk)
    static constexpr int P1LANES = (NT / SUB) >= 32 ? 1 : 32 / (NT / SUB);
    static constexpr int P2LANES = SUB < 8 ? SUB : 8;
};

// float2 entries between the exchange regions of two lines of a CTA.  `lanes` = how many different lines the 32
// lanes of a warp touch in one shared-memory instruction; the extra 256/lanes bytes de-phase their banks.
__host__ __device__ constexpr int region_stride(int rows, int lanes) {
    return ((rows * C * 8 + 255) / 256 * 256 + (lanes > 1 ? 256 / lanes : 0)) / 8;
}

// ------------------------------------------------------------------------------------------- pass 1
// One tile = SUB consecutive lines j2 of one chunk.  Thread (col, wk, line).
template <int LOG1, int LOG2>
__device__ __forceinline__ void p1_tile(const FftArgs& a, int chunk, int tile, float2* smem) {
    using K = Cfg<LOG1>;
    constexpr int L1 = K::L, L2 = 1 << LOG2, R0 = K::R0, R1 = K::R1, W = K::W, H = L1 / 2;
    constexpr int RS = region_stride(K::ROWS, K::P1LANES);
    const int tid = threadIdx.x;
    const int col = tid % C, wk = (tid / C) % W, line = tid / (C * W);
    const int j2 = tile * K::SUB + line;

    // ---- a1 + stage 0: the lower half of the line, multiplied by the strain -----------------------
    float2 u[R0];
    {
        const float2* bp = a.basisP + ((size_t)chunk * L2 + j2) * (size_t)(H * C) + col;
        const float2* dp = a.dsT + (size_t)j2 * H;
#pragma unroll
        for (int q = 0; q < R0 / 2; ++q) {
            const int j1 = wk + q * W;
            u[q] = cmul_conj(__ldg(dp + j1), ld_stream(bp + (size_t)j1 * C));
        }
    }
    dft_half<R0>(u);
    float2* reg = smem + line * RS;
#pragma unroll
    for (int m = 0; m < R0; ++m) reg[(wk * (R0 + 1) + m) * C + col] = u[m];
    __syncthreads();

    // ---- stage 1 + inter-pass twiddle + store -----------------------------------------------------
    // Y[n1][j2] is stored IN the chunk's beta block, at the address of beta[n1 + L1 j2]: the pass-2 item that owns
    // lines n1 reads exactly the addresses it later overwrites with beta, so no second buffer (and no buffer
    // hand-over between chunks) exists, and this tile's 1024 x C outputs are one contiguous run.
    float2* yrow = a.beta + ((size_t)chunk * (size_t)a.N + (size_t)j2 * L1) * C;
    const float2* tn = a.twN + (size_t)j2 * L1;
#pragma unroll
    for (int bb = 0; bb < R0 / R1; ++bb) {
        const int b = wk + bb * W;   // butterfly index < R0
        float2 x[R1];
#pragma unroll
        for (int q = 0; q < R1; ++q) x[q] = reg[(q * (R0 + 1) + b) * C + col];
#pragma unroll
        for (int q = 1; q < R1; ++q) x[q] = cmul(x[q], __ldg(a.tw1_a + q * R0 + b));
        dft<R1>(x);
#pragma unroll
        for (int m = 0; m < R1; ++m) {
            const int n1 = b + m * R0;
            const float2 v = cmul(x[m], __ldg(tn + n1));
            __stcg(yrow + n1 * C + col, v);
        }
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        atomicAdd(a.sched + 16 + chunk, 1u);
    }
}

// ------------------------------------------------------------------------------------------- pass 2
__device__ __forceinline__ void store_planes(const FftArgs& a, int bin, int gcol, float2 v) {
    if (a.plane_fp16) {
        // screen mode: one fp16 plane (round to nearest; |v| > 65504 becomes inf, which the screen lets through)
        const size_t e = ((size_t)(gcol / 32) * a.M + bin) * 64 + (gcol % 32) * 2;
        *reinterpret_cast<__half2*>(a.plane_hi + e) = __floats2half2_rn(v.x, v.y);
        return;
    }
    const __nv_bfloat16 hx = __float2bfloat16_rn(v.x), hy = __float2bfloat16_rn(v.y);
    const __nv_bfloat16 lx = __float2bfloat16_rn(v.x - __bfloat162float(hx));
    const __nv_bfloat16 ly = __float2bfloat16_rn(v.y - __bfloat162float(hy));
    const size_t e = ((size_t)(gcol / 32) * a.M + bin) * 64 + (gcol % 32) * 2;
    *reinterpret_cast<ushort2*>(a.plane_hi + e) = make_ushort2(__bfloat16_as_ushort(hx), __bfloat16_as_ushort(hy));
    *reinterpret_cast<ushort2*>(a.plane_lo + e) = make_ushort2(__bfloat16_as_ushort(lx), __bfloat16_as_ushort(ly));
}

// One item = span = max(w, SUB) consecutive lines n1 of one chunk, SUB at a time.  Thread (col, line, wk).
template <int LOG1, int LOG2>
__device__ __forceinline__ void p2_item(const FftArgs& a, int chunk, int item, float2* smem) {
    using K = Cfg<LOG2>;
    constexpr int L1 = 1 << LOG1, L2 = K::L, R0 = K::R0, R1 = K::R1, W = K::W, SUB = K::SUB;
    constexpr int RS = region_stride(K::ROWS, K::P2LANES);
    constexpr int NIT = (L2 * C + NT - 1) / NT;   // reduced outputs per thread and per group of lines
    const int tid = threadIdx.x;
    const int col = tid % C, line = (tid / C) % SUB, wk = tid / (C * SUB);
    const int w = a.w;
    const int span = w > SUB ? w : SUB;
    const int rounds = span / SUB;
    const int n1_0 = item * span;
    const int gcol = chunk * C + col;

    if (tid == 0) wait_counter(a.sched + 16 + chunk, (unsigned)(L2 / Cfg<LOG1>::SUB));
    __syncthreads();

    float2* bchunk = a.beta + (size_t)chunk * (size_t)a.N * C;   // holds Y on entry, beta on exit (in place)
    float2* reg = smem + line * RS;
    float2 acc[NIT];
#pragma unroll
    for (int i = 0; i < NIT; ++i) acc[i] = make_float2(0.f, 0.f);

    // Y loads of line n1 (stage-0 inputs).  The loads of round rd + 1 are issued as soon as u[] is free in round rd
    // (after its outputs went to shared memory for the bin sums), so their L2 latency overlaps the summation.
    float2 u[R0];
    auto load_line = [&](int n1) {
        const float2* yp = bchunk + (size_t)n1 * C + col;
#pragma unroll
        for (int q = 0; q < R0; ++q) u[q] = __ldcg(yp + (size_t)(wk + q * W) * (L1 * C));
    };
    load_line(n1_0 + line);

    for (int rd = 0; rd < rounds; ++rd) {
        const int n1 = n1_0 + rd * SUB + line;
        dft<R0>(u);
#pragma unroll
        for (int m = 0; m < R0; ++m) reg[(wk * (R0 + 1) + m) * C + col] = u[m];
        __syncthreads();
#pragma unroll
        for (int bb = 0; bb < R0 / R1; ++bb) {
            const int b = wk + bb * W;
            float2 x[R1];
#pragma unroll
            for (int q = 0; q < R1; ++q) x[q] = reg[(q * (R0 + 1) + b) * C + col];
#pragma unroll
            for (int q = 1; q < R1; ++q) x[q] = cmul(x[q], __ldg(a.tw1_b + q * R0 + b));
            dft<R1>(x);
#pragma unroll
            for (int m = 0; m < R1; ++m) {
                const int n2 = b + m * R0;
                const size_t n = (size_t)n1 + (size_t)L1 * n2;
                __stcs(bchunk + n * C + col, x[m]);
                u[bb * R1 + m] = x[m];
            }
        }
        // ---- a3: sum the outputs of gs = min(w, SUB) consecutive lines at equal n2 ------------------------
        __syncthreads();   // every stage-1 read of the exchange regions is done
#pragma unroll
        for (int bb = 0; bb < R0 / R1; ++bb)
#pragma unroll
            for (int m = 0; m < R1; ++m) reg[((wk + bb * W) + m * R0) * C + col] = u[bb * R1 + m];
        if (rd + 1 < rounds) load_line(n1 + SUB);
        __syncthreads();
        if (w >= SUB) {
            // all SUB lines of this round fall into one bin per n2; a bin spans `rounds` rounds
#pragma unroll
            for (int it = 0; it < NIT; ++it) {
                const int e = tid + it * NT;   // (n2, col): col is this thread's own
                if (L2 * C >= NT || e < L2 * C) {
                    const int n2 = e / C;
                    float2 sum = smem[n2 * C + col];
#pragma unroll
                    for (int rr = 1; rr < SUB; ++rr) sum = cadd(sum, smem[rr * RS + n2 * C + col]);
                    acc[it] = cadd(acc[it], sum);
                    if (rd == rounds - 1)
                        store_planes(a, n1_0 / w + (L1 / w) * n2, gcol,
                                     make_float2(acc[it].x * a.inv_w, acc[it].y * a.inv_w));
                }
            }
        } else {
            // w < SUB (including w = 1): this round completes SUB / w bins per n2; compact, not unrolled
            const int nb = SUB / w;
#pragma unroll 1
            for (int e = tid; e < nb * L2 * C; e += NT) {
                const int rb = e / (L2 * C), n2 = (e % (L2 * C)) / C;
                float2 sum = smem[(rb * w) * RS + n2 * C + col];
#pragma unroll 1
                for (int rr = 1; rr < w; ++rr) sum = cadd(sum, smem[(rb * w + rr) * RS + n2 * C + col]);
                store_planes(a, (n1_0 + rd * SUB + rb * w) / w + (L1 / w) * n2, gcol,
                             make_float2(sum.x * a.inv_w, sum.y * a.inv_w));
            }
        }
        __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------- kernel
template <int LOG1, int LOG2>
constexpr size_t fused_smem_bytes() {
    using K1 = Cfg<LOG1>;
    using K2 = Cfg<LOG2>;
    const size_t s1 = (size_t)K1::SUB * region_stride(K1::ROWS, K1::P1LANES) * 8;
    const size_t s2 = (size_t)K2::SUB * region_stride(K2::ROWS, K2::P2LANES) * 8;
    return s1 > s2 ? s1 : s2;
}

template <int LOG1, int LOG2>
__global__ void __launch_bounds__(NT, 2) fft_fused_kernel(const FftArgs a) {
    extern __shared__ __align__(16) float2 smem[];
    __shared__ int s_next[2];
    constexpr int L1 = 1 << LOG1, L2 = 1 << LOG2;
    const int n1t = L2 / Cfg<LOG1>::SUB;                                      // pass-1 tiles per chunk
    const int span = a.w > Cfg<LOG2>::SUB ? a.w : Cfg<LOG2>::SUB;
    const int n2t = L1 / span;                                                // pass-2 items per chunk
    const int per = n1t + n2t;
    const int total = a.nchunk * per;

    if (threadIdx.x == 0) s_next[0] = (int)atomicAdd(a.sched, 1u);
    __syncthreads();
    int t = s_next[0];
    for (int it = 0; t < total; ++it) {
        // draw the next ticket early; every tile has a barrier between this write and the read below
        if (threadIdx.x == 0) s_next[(it + 1) & 1] = (int)atomicAdd(a.sched, 1u);
        // queue order: P1(0) | P1(1) P2(0) | P1(2) P2(1) | ... | P1(n-1) P2(n-2) | P2(n-1)
        int chunk = 0, idx = t;
        bool first = true;
        if (t >= n1t) {
            const int u = t - n1t;
            const int blk = u / per, v = u - blk * per;
            if (blk < a.nchunk - 1 && v < n1t) { chunk = blk + 1; idx = v; }
            else { first = false; chunk = blk; idx = blk < a.nchunk - 1 ? v - n1t : v; }
        }
        if (first) p1_tile<LOG1, LOG2>(a, chunk, idx, smem);
        else p2_item<LOG1, LOG2>(a, chunk, idx, smem);
        t = s_next[(it + 1) & 1];
    }
}

template <int LOG1, int LOG2>
cudaError_t configure_one(int* ctas_per_sm, size_t* smem_bytes) {
    constexpr size_t smem = fused_smem_bytes<LOG1, LOG2>();
    cudaError_t e = cudaFuncSetAttribute(fft_fused_kernel<LOG1, LOG2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)smem);
    if (e != cudaSuccess) return e;
    int n = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, fft_fused_kernel<LOG1, LOG2>, NT, smem);
    if (e != cudaSuccess) return e;
    *ctas_per_sm = n;
    *smem_bytes = smem;
    return cudaSuccess;
}

template <int LOG1, int LOG2>
cudaError_t launch_one(const FftArgs& a, int grid, cudaStream_t st) {
    fft_fused_kernel<LOG1, LOG2><<<grid, NT, fused_smem_bytes<LOG1, LOG2>(), st>>>(a);
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

cudaError_t fft_fused_configure(int logL1, int logL2, int* ctas_per_sm, size_t* smem_bytes) {
    RBMF_FFT_DISPATCH(configure_one, ctas_per_sm, smem_bytes)
}

cudaError_t launch_fft_fused(const FftArgs& a, int logL1, int logL2, int grid, cudaStream_t st) {
    RBMF_FFT_DISPATCH(launch_one, a, grid, st)
}

}  // namespace rbmf
