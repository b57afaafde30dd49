// Kernel 1: pointwise correlation fused into a batched Stockham inverse FFT (steps a1-a3 of include/rbmf.h).
//
// Layout: every array is "time/frequency-major, basis-column contiguous": element (row, c) of an R x k array is at
// row*k + c.  The FFT runs along the row index for each of the k columns independently ("batch-innermost"), so a
// butterfly input is a run of kFftKC consecutive columns = one 64-byte segment, at any row stride.
//
// Length N = L1 * L2 is done in two passes through HBM (four-step FFT):
//   pass 1 (one CTA per j2, L = L1):   Y[n1][j2] = e^{2 pi i j2 n1 / N} sum_{j1} G[j1 L2 + j2] e^{2 pi i j1 n1 / L1}
//   pass 2 (one CTA per n1, L = L2):   beta[n1 + L1 n2] = sum_{j2} Y[n1][j2] e^{2 pi i j2 n2 / L2}
// with G[j] = s d[j] conj(b[j]) formed in registers by pass 1's loads (never stored).
// beta^avg (Eq. 9) is obtained as the paper's Eq. 10-12 states: the w-sample bin
// average equals a length-N/w inverse FFT of the alias-folded spectrum Omega(f') = sum_l G[l N/w + f'] S(l N/w + f');
// pass 1 in "fold" mode forms Omega in registers from the same basis rows, and pass 2 in "planes" mode writes the
// result directly as the bf16 hi/lo operand planes of kernel 2.
//
// Inside a CTA a length-L transform is 2 or 3 radix-8/16 Stockham stages; data stays in registers across the
// butterflies and is exchanged between stages through (padded) shared memory.
#include <cuda_bf16.h>

#include "rbmf_internal.h"

namespace rbmf {

namespace {

constexpr int KC = kFftKC;

template <int LOGL> struct FftCfg;
template <> struct FftCfg<5>  { static constexpr int NS = 2, R0 = 8,  R1 = 4,  R2 = 1, EPT = 8;  };
template <> struct FftCfg<6>  { static constexpr int NS = 2, R0 = 8,  R1 = 8,  R2 = 1, EPT = 8;  };
template <> struct FftCfg<7>  { static constexpr int NS = 2, R0 = 16, R1 = 8,  R2 = 1, EPT = 16; };
template <> struct FftCfg<8>  { static constexpr int NS = 2, R0 = 16, R1 = 16, R2 = 1, EPT = 16; };
template <> struct FftCfg<9>  { static constexpr int NS = 3, R0 = 8,  R1 = 8,  R2 = 8, EPT = 8;  };
template <> struct FftCfg<10> { static constexpr int NS = 3, R0 = 16, R1 = 8,  R2 = 8, EPT = 16; };

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cmul_conj(float2 d, float2 b) {   // d * conj(b)
    return make_float2(d.x * b.x + d.y * b.y, d.y * b.x - d.x * b.y);
}

// v * e^{+2 pi i m / 16}, 0 <= m < 8; m is a compile-time constant after unrolling.
__device__ __forceinline__ float2 mul_w16(float2 v, int m) {
    constexpr float C1 = 0.92387953251128674f, C2 = 0.70710678118654752f, C3 = 0.38268343236508977f;
    switch (m) {
        case 0: return v;
        case 1: return cmul(v, make_float2(C1, C3));
        case 2: return make_float2((v.x - v.y) * C2, (v.x + v.y) * C2);
        case 3: return cmul(v, make_float2(C3, C1));
        case 4: return make_float2(-v.y, v.x);
        case 5: return cmul(v, make_float2(-C3, C1));
        case 6: return make_float2((-v.x - v.y) * C2, (v.x - v.y) * C2);
        default: return cmul(v, make_float2(-C1, C3));
    }
}

// In-register inverse DFT of length R (natural order in and out): x[m] <- sum_j x[j] e^{+2 pi i j m / R}.
template <int R>
__device__ __forceinline__ void dft(float2 (&x)[R]) {
    if constexpr (R == 2) {
        const float2 a = x[0], b = x[1];
        x[0] = make_float2(a.x + b.x, a.y + b.y);
        x[1] = make_float2(a.x - b.x, a.y - b.y);
    } else {
        float2 e[R / 2], o[R / 2];
#pragma unroll
        for (int i = 0; i < R / 2; ++i) { e[i] = x[2 * i]; o[i] = x[2 * i + 1]; }
        dft<R / 2>(e);
        dft<R / 2>(o);
#pragma unroll
        for (int i = 0; i < R / 2; ++i) {
            const float2 t = mul_w16(o[i], i * (16 / R));
            x[i] = make_float2(e[i].x + t.x, e[i].y + t.y);
            x[i + R / 2] = make_float2(e[i].x - t.x, e[i].y - t.y);
        }
    }
}

// One Stockham stage on the thread's EPT elements: EPT/R butterflies of radix R; NSB = product of earlier radices.
template <int L, int R, int EPT, int NSB>
__device__ __forceinline__ void twiddle_and_dft(float2 (&u)[EPT], int wk, const float2* __restrict__ tw) {
    constexpr int NB = EPT / R;
    constexpr int W = L / EPT;
#pragma unroll
    for (int bb = 0; bb < NB; ++bb) {
        float2 x[R];
#pragma unroll
        for (int q = 0; q < R; ++q) x[q] = u[bb * R + q];
        if constexpr (NSB > 1) {
            const int b = wk + bb * W;
            const int i1 = (b & (NSB - 1)) * (L / (NSB * R));
            float2 wq[R];
            wq[0] = make_float2(1.f, 0.f);
            wq[1] = __ldg(tw + i1);
            if constexpr (R >= 4) { wq[2] = __ldg(tw + 2 * i1); wq[3] = cmul(wq[1], wq[2]); }
            if constexpr (R >= 8) {
                wq[4] = __ldg(tw + 4 * i1);
#pragma unroll
                for (int q = 1; q < 4; ++q) wq[4 + q] = cmul(wq[q], wq[4]);
            }
            if constexpr (R >= 16) {
                wq[8] = __ldg(tw + 8 * i1);
#pragma unroll
                for (int q = 1; q < 8; ++q) wq[8 + q] = cmul(wq[q], wq[8]);
            }
#pragma unroll
            for (int q = 1; q < R; ++q) x[q] = cmul(x[q], wq[q]);
        }
        dft<R>(x);
#pragma unroll
        for (int q = 0; q < R; ++q) u[bb * R + q] = x[q];
    }
}

__device__ __forceinline__ int pad_row(int r) { return r + (r >> 4); }

enum : int { P1_MAIN = 0, P1_FOLD = 1, P2_BETA = 2, P2_PLANES = 3, P2_BOTH = 4 };

template <int L, int MODE>
__device__ __forceinline__ float2 load_elem(const FftArgs& a, int l, int o, int col) {
    if constexpr (MODE == P1_MAIN) {
        const int j = l * a.lines + o;
        if (j < a.j_low || j >= a.n_half) return make_float2(0.f, 0.f);
        return cmul_conj(__ldg(a.strain + j), __ldg(a.in + (size_t)j * a.k + col));
    } else if constexpr (MODE == P1_FOLD) {
        float2 acc = make_float2(0.f, 0.f);
        int j = l * a.lines + o;
        for (int r = 0; r < a.fold; ++r, j += a.fold_stride) {
            if (j >= a.j_low && j < a.n_half) {
                const float2 t = cmul_conj(__ldg(a.strain + j), __ldg(a.in + (size_t)j * a.k + col));
                acc.x += t.x;
                acc.y += t.y;
            }
        }
        return acc;
    } else {
        return __ldg(a.in + ((size_t)o * L + l) * a.k + col);
    }
}

__device__ __forceinline__ void store_planes(const FftArgs& a, size_t row, int col, float2 v) {
    const __nv_bfloat16 hx = __float2bfloat16_rn(v.x), hy = __float2bfloat16_rn(v.y);
    const __nv_bfloat16 lx = __float2bfloat16_rn(v.x - __bfloat162float(hx));
    const __nv_bfloat16 ly = __float2bfloat16_rn(v.y - __bfloat162float(hy));
    const size_t e = row * (size_t)(2 * a.k) + 2 * col;
    *reinterpret_cast<ushort2*>(a.plane_hi + e) = make_ushort2(__bfloat16_as_ushort(hx), __bfloat16_as_ushort(hy));
    *reinterpret_cast<ushort2*>(a.plane_lo + e) = make_ushort2(__bfloat16_as_ushort(lx), __bfloat16_as_ushort(ly));
}

template <int L, int MODE>
__device__ __forceinline__ void store_elem(const FftArgs& a, int l, int o, int col, float2 v) {
    if constexpr (MODE == P1_MAIN || MODE == P1_FOLD) {
        const int m = o * l;   // < Ntot <= 2^20
        const float2 t = cmul(__ldg(a.tw_hi + (m >> 10)), __ldg(a.tw_lo + (m & 1023)));
        a.out[((size_t)l * a.lines + o) * a.k + col] = cmul(v, t);
    } else {
        const size_t row = (size_t)o + (size_t)a.lines * l;
        if constexpr (MODE == P2_BETA || MODE == P2_BOTH) a.out[row * a.k + col] = v;
        if constexpr (MODE == P2_PLANES || MODE == P2_BOTH) store_planes(a, row, col, v);
    }
}

template <int LOGL, int MODE>
__global__ void __launch_bounds__((1 << LOGL) * KC / FftCfg<LOGL>::EPT)
fft_pass_kernel(const FftArgs a) {
    using Cfg = FftCfg<LOGL>;
    constexpr int L = 1 << LOGL, EPT = Cfg::EPT, W = L / EPT;
    constexpr int R0 = Cfg::R0, R1 = Cfg::R1, R2 = Cfg::R2;
    extern __shared__ float2 sm[];   // (L + L/16) rows x KC columns

    const int c = threadIdx.x % KC, wk = threadIdx.x / KC;
    // Column chunks are the fastest-varying block index: the CTAs that touch the two 64-byte halves of one 128-byte
    // line run at the same time, so the second half is an L2 hit instead of a second DRAM fetch.
    const int o = blockIdx.y;
    const int col = blockIdx.x * KC + c;
    const float2* __restrict__ tw = a.tw_L;
    float2 u[EPT];

    // ---- stage 0: straight from global memory ------------------------------------------------
#pragma unroll
    for (int bb = 0; bb < EPT / R0; ++bb)
#pragma unroll
        for (int q = 0; q < R0; ++q)
            u[bb * R0 + q] = load_elem<L, MODE>(a, (wk + bb * W) + q * (L / R0), o, col);
    twiddle_and_dft<L, R0, EPT, 1>(u, wk, tw);
#pragma unroll
    for (int bb = 0; bb < EPT / R0; ++bb)
#pragma unroll
        for (int q = 0; q < R0; ++q)
            sm[pad_row((wk + bb * W) * R0 + q) * KC + c] = u[bb * R0 + q];
    __syncthreads();

    // ---- stage 1 -----------------------------------------------------------------------------
#pragma unroll
    for (int bb = 0; bb < EPT / R1; ++bb)
#pragma unroll
        for (int q = 0; q < R1; ++q)
            u[bb * R1 + q] = sm[pad_row((wk + bb * W) + q * (L / R1)) * KC + c];
    twiddle_and_dft<L, R1, EPT, R0>(u, wk, tw);
    if constexpr (Cfg::NS == 2) {
#pragma unroll
        for (int bb = 0; bb < EPT / R1; ++bb)
#pragma unroll
            for (int q = 0; q < R1; ++q)
                store_elem<L, MODE>(a, (wk + bb * W) + q * (L / R1), o, col, u[bb * R1 + q]);
    } else {
        __syncthreads();
#pragma unroll
        for (int bb = 0; bb < EPT / R1; ++bb) {
            const int b = wk + bb * W;
            const int j0 = (b / R0) * (R0 * R1) + (b % R0);
#pragma unroll
            for (int q = 0; q < R1; ++q) sm[pad_row(j0 + q * R0) * KC + c] = u[bb * R1 + q];
        }
        __syncthreads();
        // ---- stage 2 -------------------------------------------------------------------------
#pragma unroll
        for (int bb = 0; bb < EPT / R2; ++bb)
#pragma unroll
            for (int q = 0; q < R2; ++q)
                u[bb * R2 + q] = sm[pad_row((wk + bb * W) + q * (L / R2)) * KC + c];
        twiddle_and_dft<L, R2, EPT, R0 * R1>(u, wk, tw);
#pragma unroll
        for (int bb = 0; bb < EPT / R2; ++bb)
#pragma unroll
            for (int q = 0; q < R2; ++q)
                store_elem<L, MODE>(a, (wk + bb * W) + q * (L / R2), o, col, u[bb * R2 + q]);
    }
}

template <int LOGL, int MODE>
cudaError_t launch_one(const FftArgs& a, cudaStream_t st) {
    constexpr int L = 1 << LOGL;
    constexpr int NT = L * KC / FftCfg<LOGL>::EPT;
    constexpr size_t smem = (size_t)(L + L / 16) * KC * sizeof(float2);
    static bool configured = false;
    if (!configured && smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(fft_pass_kernel<LOGL, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    dim3 grid((unsigned)(a.k / KC), (unsigned)a.lines);
    fft_pass_kernel<LOGL, MODE><<<grid, NT, smem, st>>>(a);
    return cudaGetLastError();
}

template <int MODE>
cudaError_t dispatch(const FftArgs& a, int logL, cudaStream_t st) {
    switch (logL) {
        case 5: return launch_one<5, MODE>(a, st);
        case 6: return launch_one<6, MODE>(a, st);
        case 7: return launch_one<7, MODE>(a, st);
        case 8: return launch_one<8, MODE>(a, st);
        case 9: return launch_one<9, MODE>(a, st);
        case 10: return launch_one<10, MODE>(a, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

cudaError_t launch_fft_pass1(const FftArgs& a, int logL, bool fold, cudaStream_t st) {
    return fold ? dispatch<P1_FOLD>(a, logL, st) : dispatch<P1_MAIN>(a, logL, st);
}

cudaError_t launch_fft_pass2(const FftArgs& a, int logL, int mode, cudaStream_t st) {
    switch (mode) {
        case 0: return dispatch<P2_BETA>(a, logL, st);
        case 1: return dispatch<P2_PLANES>(a, logL, st);
        case 2: return dispatch<P2_BOTH>(a, logL, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace rbmf
