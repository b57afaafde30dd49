// Set-up kernels: constant tables, basis re-layout, coefficient planes, per-call strain scaling.
// None of them is on the per-segment critical path except prep_strain (N/2 elements).
#include <cuda_bf16.h>
#include <cuda_fp16.h>

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

// tw1[q * R0 + b] = e^{2 pi i q b / L} (stage-1 twiddles of a length-L = R0 * R1 line, q < R1, b < R0);
// Inter-pass twiddles of the four-step FFT, e^{2 pi i j2 n1 / N} with n1 = b + m R0 (b < R0, m < R1), as two small
// tables whose product they are:  twN[j2 * R0 + b] = e^{2 pi i j2 b / N}  (L2 x R0 entries), followed by
// twN[L2 * R0 + j2 * R1 + m] = e^{2 pi i j2 m R0 / N}  (L2 x R1 entries): 256 KB instead of N entries.
__global__ void init_tables_kernel(float2* tw1_a, float2* tw1_b, float2* twN, int logL1, int logL2) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    const int L1 = 1 << logL1, L2 = 1 << logL2;
    const long long N = (long long)L1 * L2;
    if (i < L1) { const int R0 = fft_r0(logL1); tw1_a[i] = unit_root((i / R0) * (i % R0), L1); }
    if (i < L2) { const int R0 = fft_r0(logL2); tw1_b[i] = unit_root((i / R0) * (i % R0), L2); }
    const int R0 = fft_r0(logL1), R1 = fft_r1(logL1);
    if (i < (long long)L2 * R0) twN[i] = unit_root((i / R0) * (i % R0), N);
    if (i < (long long)L2 * R1) twN[(long long)L2 * R0 + i] = unit_root((i / R1) * (i % R1) * R0, N);
}

cudaError_t launch_init_tables(float2* tw1_a, float2* tw1_b, float2* twN, int logL1, int logL2, cudaStream_t st) {
    const long long n = 1LL << (logL1 + logL2);
    const int threads = 256;
    init_tables_kernel<<<(unsigned)((n + threads - 1) / threads), threads, 0, st>>>(tw1_a, tw1_b, twN, logL1, logL2);
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------- basis re-layout
// basis: k x bins (row-major, caller's layout)  ->  basisP[chunk][tile][j1 < L1/2][line < sub][C] with
// j = j1 L2 + j2, j2 = tile * sub + line, zero outside the band: the block a pass-1 tile (sub lines) reads is
// contiguous and already in the [position][line][column] order of the FFT kernel's tile buffer.
// Rows >= rows_valid (the padding of the last slab of a template bank, template_route.cu) are written as zeros.
__global__ void layout_basis_kernel(const float2* __restrict__ basis, float2* __restrict__ basisP, long long bins,
                                    int j_low, int logL1, int logL2, int sub, int rows_valid) {
    __shared__ float2 tile[kFftC][32][33];
    const int L2 = 1 << logL2, H = (1 << logL1) / 2;
    const int chunk = blockIdx.z;
    const int j2_0 = blockIdx.x * 32, j1_0 = blockIdx.y * 32;
    const int tx = threadIdx.x % 32, ty = threadIdx.x / 32;   // 32 x 8
    for (int c = 0; c < kFftC; ++c)
        for (int r = ty; r < 32; r += 8) {
            const int j1 = j1_0 + r, j2 = j2_0 + tx;
            float2 v = make_float2(0.f, 0.f);
            if (j1 < H && j2 < L2) {
                const long long j = (long long)j1 * L2 + j2;
                if (j >= j_low && chunk * kFftC + c < rows_valid) v = basis[(long long)(chunk * kFftC + c) * bins + j];
            }
            tile[c][r][tx] = v;
        }
    __syncthreads();
    // write: for each j2 of the tile, 32 j1 x C columns are contiguous
    for (int r = ty; r < 32; r += 8) {
        const int j2 = j2_0 + r;
        if (j2 >= L2) continue;
        for (int e = tx; e < 32 * kFftC; e += 32) {
            const int j1 = j1_0 + e / kFftC, c = e % kFftC;
            if (j1 < H)
                basisP[((((size_t)chunk * (L2 / sub) + j2 / sub) * fft_p1_rows(logL1) + fft_p1_row(logL1, j1)) * sub +
                        j2 % sub) * kFftC + c] = tile[c][e / kFftC][r];
        }
    }
}

cudaError_t launch_layout_basis(const float2* basis, float2* basisP, int k, int64_t bins, int j_low, int logL1,
                                int logL2, int sub, int rows_valid, cudaStream_t st) {
    const int L2 = 1 << logL2, H = (1 << logL1) / 2;
    dim3 grid((unsigned)((L2 + 31) / 32), (unsigned)((H + 31) / 32), (unsigned)(k / kFftC));
    layout_basis_kernel<<<grid, 256, 0, st>>>(basis, basisP, bins, j_low, logL1, logL2, sub, rows_valid);
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

// Screen mode (RBMF_GEMM_SCREEN) additionally needs the same two rows rounded ONCE to fp16 (c_h16) and, per block of
// 128 templates, tnorm_blk[tb] = max_t ||c_t||_2 / sigma_t (fp32 values as stored in cs; zero-initialised by the
// launcher, positive floats order like their bit patterns so atomicMax on the bits is exact).
__global__ void prep_coeffs_kernel(const float2* __restrict__ coeffs, const float* __restrict__ sigma,
                                   float2* __restrict__ cs, uint16_t* __restrict__ c_hi,
                                   uint16_t* __restrict__ c_lo, uint16_t* __restrict__ c_h16,
                                   float* __restrict__ tnorm_blk, int T, int k) {
    const int t = blockIdx.x;
    const int tb = t / kGemmTT, r = t % kGemmTT;
    const size_t row_re = ((size_t)tb * 2 * kGemmTT + r) * (size_t)(2 * k);
    const size_t row_im = ((size_t)tb * 2 * kGemmTT + kGemmTT + r) * (size_t)(2 * k);
    if (t >= T) {
        for (int c = threadIdx.x; c < 2 * k; c += blockDim.x) {
            c_hi[row_re + c] = 0; c_lo[row_re + c] = 0; c_h16[row_re + c] = 0;
            c_hi[row_im + c] = 0; c_lo[row_im + c] = 0; c_h16[row_im + c] = 0;
        }
        return;
    }
    __shared__ double red[32];
    __shared__ double red2[32];
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
        const float sg = sigma[t];
        inv_sigma = (sg > 0.f && sg <= 3.0e38f) ? 1.0f / sg : 0.f;   // not a positive finite norm: template disabled
    }
    __syncthreads();
    const float is = inv_sigma;
    double nsq = 0.0;
    for (int c = threadIdx.x; c < k; c += blockDim.x) {
        const float2 v = coeffs[(size_t)t * k + c];
        const float a = v.x * is, b = v.y * is;
        nsq += (double)a * a + (double)b * b;
        cs[(size_t)t * k + c] = make_float2(a, -b);   // conj(c)/sigma for stage 2
        {
            const uint16_t ha = __half_as_ushort(__float2half_rn(a)), hb = __half_as_ushort(__float2half_rn(b));
            c_h16[row_re + 2 * c] = ha;     c_h16[row_re + 2 * c + 1] = hb;
            c_h16[row_im + 2 * c] = hb ^ 0x8000u; c_h16[row_im + 2 * c + 1] = ha;
        }
        uint16_t h, l;
        split_bf16(a, h, l);
        c_hi[row_re + 2 * c] = h;     c_lo[row_re + 2 * c] = l;
        c_hi[row_im + 2 * c + 1] = h; c_lo[row_im + 2 * c + 1] = l;
        split_bf16(b, h, l);
        c_hi[row_re + 2 * c + 1] = h; c_lo[row_re + 2 * c + 1] = l;
        split_bf16(-b, h, l);
        c_hi[row_im + 2 * c] = h;     c_lo[row_im + 2 * c] = l;
    }
    for (int o = 16; o > 0; o >>= 1) nsq += __shfl_xor_sync(0xffffffffu, nsq, o);
    if ((threadIdx.x & 31) == 0) red2[threadIdx.x >> 5] = nsq;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s2 = 0.0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) s2 += red2[i];
        const float nt = (float)(sqrt(s2) * (1.0 + 1e-6));
        atomicMax(reinterpret_cast<unsigned*>(tnorm_blk + tb), __float_as_uint(nt));
    }
}

cudaError_t launch_prep_coeffs(const float2* coeffs, const float* sigma, float2* cs, uint16_t* c_hi,
                               uint16_t* c_lo, uint16_t* c_h16, float* tnorm_blk, int T, int Tpad, int k,
                               cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(tnorm_blk, 0, (size_t)(Tpad / kGemmTT) * sizeof(float), st);
    if (e != cudaSuccess) return e;
    prep_coeffs_kernel<<<Tpad, 128, 0, st>>>(coeffs, sigma, cs, c_hi, c_lo, c_h16, tnorm_blk, T, k);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------ per-bin norms (screen mode)
// bin_norm[i] >= ||beta^avg[i]||_2 over the k columns, from the fp16 plane [kb][bin][64]: the stored values are
// within 2^-11 relative (+ 2^-25 absolute in the subnormal range) of the fp32 ones, hence the inflation.
// Eight lanes share a bin (16 bytes each of its 128-byte K-block row); consecutive lanes read consecutive bytes.
__global__ void __launch_bounds__(256) bin_norm_kernel(const uint16_t* __restrict__ plane, float* __restrict__ bin_norm,
                                                       int M, int Mplane, int nkb) {
    const long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long bin = gid >> 3;
    const int piece = (int)(gid & 7);
    float acc = 0.f;
    if (bin < M) {
        const uint4* p = reinterpret_cast<const uint4*>(plane) + bin * 8 + piece;
        for (int kb = 0; kb < nkb; ++kb) {
            const uint4 v = __ldg(p + (size_t)kb * Mplane * 8);
            const unsigned wds[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const float2 f = __half22float2(*reinterpret_cast<const __half2*>(&wds[i]));
                acc = fmaf(f.x, f.x, acc);
                acc = fmaf(f.y, f.y, acc);
            }
        }
    }
    acc += __shfl_xor_sync(0xffffffffu, acc, 1);
    acc += __shfl_xor_sync(0xffffffffu, acc, 2);
    acc += __shfl_xor_sync(0xffffffffu, acc, 4);
    if (bin < M && piece == 0) bin_norm[bin] = sqrtf(acc) * (1.0f + 0x1p-9f) + 1e-5f;
}

// M = bins to process (all segments of the batch), Mplane = rows of the plane (its K-block stride)
cudaError_t launch_bin_norm(const uint16_t* plane_h16, float* bin_norm, int M, int Mplane, int nkb, cudaStream_t st) {
    const long long threads = (long long)M * 8;
    bin_norm_kernel<<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(plane_h16, bin_norm, M, Mplane, nkb);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------ strain prep
// dsT[b][j2][j1] = s d_b[j1 L2 + j2], j1 < L1/2 (s = sqrt(2/N)): the strain of segment b (blockIdx.y;
// N/2 + 1 bins per segment on input) in the order pass 1 of the FFT reads it.
__global__ void prep_strain_kernel(const float2* __restrict__ strain, float2* __restrict__ dsT, int logL1,
                                   int logL2, float scale) {
    const int L2 = 1 << logL2, H = (1 << logL1) / 2;
    const int j = blockIdx.x * blockDim.x + threadIdx.x;   // j = j1 L2 + j2 < N/2
    if (j >= H * L2) return;
    const float2 d = strain[(size_t)blockIdx.y * ((size_t)H * L2 + 1) + j];
    const size_t row = (size_t)fft_strain_row(logL1);
    dsT[((size_t)blockIdx.y * L2 + (size_t)(j % L2)) * row + j / L2] = make_float2(d.x * scale, d.y * scale);
}

cudaError_t launch_prep_strain(const float2* strain, float2* dsT, int logL1, int logL2, float scale, int nb,
                               cudaStream_t st) {
    const int n_half = 1 << (logL1 + logL2 - 1);
    prep_strain_kernel<<<dim3((n_half + 255) / 256, nb), 256, 0, st>>>(strain, dsT, logL1, logL2, scale);
    return cudaGetLastError();
}

}  // namespace rbmf
