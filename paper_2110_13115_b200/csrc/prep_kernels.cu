// Set-up kernels: constant tables, basis transpose, coefficient planes, per-call strain scaling.
// None of them is on the per-segment critical path except prep_strain (N/2 elements).
#include <cuda_bf16.h>

#include "rbmf_internal.h"

namespace rbmf {

// --------------------------------------------------------------------------------------- tables
// Twiddles are evaluated in fp64 (sincospi on exact rational arguments) and stored as fp32:
// "twiddles from an exact table, never __sincosf" (hard parts).
__device__ __forceinline__ float2 unit_root(long long num, long long den) {
    // e^{2 pi i num/den}
    double s, c;
    sincospi(2.0 * (double)(num % den) / (double)den, &s, &c);
    return make_float2((float)c, (float)s);
}

__global__ void init_tables_kernel(float2* tw_L_all, float2* tw_lo_main, float2* tw_hi_main, float2* tw_lo_avg,
                                   float2* tw_hi_avg, float2* S_table, long long N, long long M, int w) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    // per-length tables, L = 32 .. 1024
    if (i < kTwAllEntries) {
        for (int logL = 5; logL <= 10; ++logL) {
            const int L = 1 << logL;
            const int off = tw_table_offset(logL);
            if (i >= off && i < off + L) tw_L_all[i] = unit_root(i - off, L);
        }
    }
    if (i < 1024) {
        tw_lo_main[i] = unit_root(i, N);
        tw_lo_avg[i] = unit_root(i, M);
    }
    const long long nh_main = N / 1024 > 0 ? N / 1024 : 1;
    const long long nh_avg = M / 1024 > 0 ? M / 1024 : 1;
    if (i < nh_main) tw_hi_main[i] = unit_root(i * 1024, N);
    if (i < nh_avg) tw_hi_avg[i] = unit_root(i * 1024, M);
    // S(j) = (1/w) sum_{r<w} e^{2 pi i j r / N}: the frequency response of the w-sample bin average
    // (Eq. 10-11, :199-208); used to obtain beta^avg as a length-N/w inverse FFT (Eq. 12).
    if (i < N / 2) {
        double sr = 0.0, si = 0.0;
        for (int r = 0; r < w; ++r) {
            double s, c;
            sincospi(2.0 * (double)((i * r) % N) / (double)N, &s, &c);
            sr += c;
            si += s;
        }
        S_table[i] = make_float2((float)(sr / w), (float)(si / w));
    }
}

cudaError_t launch_init_tables(float2* tw_L_all, float2* tw_lo_main, float2* tw_hi_main, float2* tw_lo_avg,
                               float2* tw_hi_avg, float2* S_table, int64_t N, int64_t M, int w, cudaStream_t st) {
    long long n = N / 2 > 2048 ? N / 2 : 2048;
    const int threads = 256;
    init_tables_kernel<<<(unsigned)((n + threads - 1) / threads), threads, 0, st>>>(
        tw_L_all, tw_lo_main, tw_hi_main, tw_lo_avg, tw_hi_avg, S_table, N, M, w);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------ basis transpose
// basis: k x bins (row-major, caller's layout)  ->  basisT: (N/2) x k, zero outside the band.
__global__ void transpose_basis_kernel(const float2* __restrict__ basis, float2* __restrict__ basisT, int k,
                                       long long bins, int j_low, int n_half) {
    __shared__ float2 tile[32][33];
    const long long j0 = (long long)blockIdx.x * 32;
    const int c0 = blockIdx.y * 32;
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const int c = c0 + r;
        const long long j = j0 + threadIdx.x;
        float2 v = make_float2(0.f, 0.f);
        if (c < k && j >= j_low && j < n_half) v = basis[(long long)c * bins + j];
        tile[r][threadIdx.x] = v;
    }
    __syncthreads();
    for (int r = threadIdx.y; r < 32; r += blockDim.y) {
        const long long j = j0 + r;
        const int c = c0 + threadIdx.x;
        if (c < k && j < n_half) basisT[j * k + c] = tile[threadIdx.x][r];
    }
}

cudaError_t launch_transpose_basis(const float2* basis, float2* basisT, int k, int64_t bins, int j_low,
                                   int n_half, cudaStream_t st) {
    dim3 grid((unsigned)((n_half + 31) / 32), (unsigned)((k + 31) / 32));
    dim3 block(32, 8);
    transpose_basis_kernel<<<grid, block, 0, st>>>(basis, basisT, k, bins, j_low, n_half);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------- coefficient planes
// For template t (block tb = t/128, r = t%128) the GEMM's B operand holds two K-major rows of 2k reals:
//   row tb*256 + r        ("re"):  ( a_0,  b_0,  a_1,  b_1, ...) / sigma_t
//   row tb*256 + 128 + r  ("im"):  (-b_0,  a_0, -b_1,  a_1, ...) / sigma_t         c_tk = a_k + i b_k
// so that  re . (x_0, y_0, ...) = Re sum_k conj(c_tk) beta_k  and  im . (...) = Im (...)  (Eq. 7),
// each split into bf16 hi + lo.  Rows of padding templates (t >= T) are zero.
__device__ __forceinline__ void split_bf16(float v, uint16_t& hi, uint16_t& lo) {
    const __nv_bfloat16 h = __float2bfloat16_rn(v);
    const __nv_bfloat16 l = __float2bfloat16_rn(v - __bfloat162float(h));
    hi = __bfloat16_as_ushort(h);
    lo = __bfloat16_as_ushort(l);
}

__global__ void prep_coeffs_kernel(const float2* __restrict__ coeffs, const float* __restrict__ sigma,
                                   float2* __restrict__ cs, uint16_t* __restrict__ c_hi,
                                   uint16_t* __restrict__ c_lo, int T, int k) {
    const int t = blockIdx.x;
    const int tb = t / kGemmTT, r = t % kGemmTT;
    const size_t row_re = ((size_t)tb * 2 * kGemmTT + r) * (size_t)(2 * k);
    const size_t row_im = ((size_t)tb * 2 * kGemmTT + kGemmTT + r) * (size_t)(2 * k);
    if (t >= T) {
        for (int c = threadIdx.x; c < 2 * k; c += blockDim.x) {
            c_hi[row_re + c] = 0; c_lo[row_re + c] = 0;
            c_hi[row_im + c] = 0; c_lo[row_im + c] = 0;
        }
        return;
    }
    __shared__ double red[32];
    __shared__ float inv_sigma;
    if (sigma == nullptr) {
        double acc = 0.0;
        for (int c = threadIdx.x; c < k; c += blockDim.x) {
            const float2 v = coeffs[(size_t)t * k + c];
            acc += (double)v.x * v.x + (double)v.y * v.y;
        }
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
        __syncthreads();
        if (threadIdx.x == 0) {
            double s = 0.0;
            for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s += red[i];
            inv_sigma = s > 0.0 ? (float)(1.0 / sqrt(s)) : 0.f;
        }
    } else if (threadIdx.x == 0) {
        inv_sigma = 1.0f / sigma[t];
    }
    __syncthreads();
    const float is = inv_sigma;
    for (int c = threadIdx.x; c < k; c += blockDim.x) {
        const float2 v = coeffs[(size_t)t * k + c];
        const float a = v.x * is, b = v.y * is;
        cs[(size_t)t * k + c] = make_float2(a, -b);   // conj(c)/sigma for stage 2
        uint16_t h, l;
        split_bf16(a, h, l);
        c_hi[row_re + 2 * c] = h;     c_lo[row_re + 2 * c] = l;
        c_hi[row_im + 2 * c + 1] = h; c_lo[row_im + 2 * c + 1] = l;
        split_bf16(b, h, l);
        c_hi[row_re + 2 * c + 1] = h; c_lo[row_re + 2 * c + 1] = l;
        split_bf16(-b, h, l);
        c_hi[row_im + 2 * c] = h;     c_lo[row_im + 2 * c] = l;
    }
}

cudaError_t launch_prep_coeffs(const float2* coeffs, const float* sigma, float2* cs, uint16_t* c_hi,
                               uint16_t* c_lo, int T, int Tpad, int k, cudaStream_t st) {
    prep_coeffs_kernel<<<Tpad, 128, 0, st>>>(coeffs, sigma, cs, c_hi, c_lo, T, k);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------ strain prep
// ds[j] = s d[j] (s = sqrt(2/N));  dS[j] = ds[j] S(j)  (alias-fold weights, Eq. 12).
__global__ void prep_strain_kernel(const float2* __restrict__ strain, const float2* __restrict__ S_table,
                                   float2* __restrict__ ds, float2* __restrict__ dS, int n_half, float scale) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_half) return;
    const float2 d = strain[j];
    const float2 v = make_float2(d.x * scale, d.y * scale);
    ds[j] = v;
    const float2 s = S_table[j];
    dS[j] = make_float2(v.x * s.x - v.y * s.y, v.x * s.y + v.y * s.x);
}

cudaError_t launch_prep_strain(const float2* strain, const float2* S_table, float2* ds, float2* dS, int n_half,
                               float scale, cudaStream_t st) {
    prep_strain_kernel<<<(n_half + 255) / 256, 256, 0, st>>>(strain, S_table, ds, dS, n_half, scale);
    return cudaGetLastError();
}

}  // namespace rbmf
