// Preparation on the GPU: from a (sub-)bank of templates
// stored row-wise, T (S x bins),
//   covariance            C = T T^H                               (S x S; "conjugate transpose", reading R5; no centering, R6)
//   its k leading eigen-   by block power (subspace) iteration with re-orthonormalisation -- the paper used Lanczos
//   vectors               (:152); any orthonormal basis of the leading subspace serves the path equally --,
//   basis                 P = orth(V^H T)                          (k x bins, orthonormal rows over the band)
//   coefficients          D = T P^H, sigma_t = ||c_t||_2           (:167-169).
// Amortised, offline work (done once per sub-bank): plain fp32 CUDA-core kernels -- one tiled complex GEMM with
// periodic fp64 flushes of its accumulators (sums run over up to 2^19 frequency bins) and classical Gram-Schmidt with
// re-orthogonalisation ("twice is enough") on row vectors -- not tensor-core code: the results are INPUTS of the hot
// path and want fp32-exact orthonormality rather than speed.
#include "rbmf_internal.h"

namespace rbmf {

namespace {

constexpr int TM = 64, TN = 64, TK = 16;

// C[i][j] = sum_{p in [p0, p1)} A[i lda + p] * op(B)[p][j],  i < M, j < N
//   NN = false:  op(B)[p][j] = conj(B[j ldb + p])      ("A B^H": both operands row-major with p contiguous)
//   NN = true:   op(B)[p][j] = B[p ldb + j]
template <bool NN>
__global__ void __launch_bounds__(256) cgemm_kernel(const float2* __restrict__ A, long long lda,
                                                    const float2* __restrict__ B, long long ldb, float2* __restrict__ C,
                                                    long long ldc, int M, int N, long long p0, long long p1) {
    __shared__ float2 sA[TK][TM + 1];
    __shared__ float2 sB[TK][TN + 1];
    // one-dimensional grid over the (row tile, column tile) pairs, column tiles fastest: M may be 2^24 templates
    // (rbmf_prepare_coeffs), far more row tiles than gridDim.y allows
    const int ntn = (N + TN - 1) / TN;
    const int i0 = (int)(blockIdx.x / ntn) * TM, j0 = (int)(blockIdx.x % ntn) * TN;
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
    float2 acc[4][4];
    double2 dacc[4][4];
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) { acc[u][v] = make_float2(0.f, 0.f); dacc[u][v] = make_double2(0.0, 0.0); }
    int since_flush = 0;
    for (long long pk = p0; pk < p1; pk += TK) {
        for (int e = threadIdx.x; e < TM * TK; e += 256) {
            const int i = e / TK, kk = e % TK;
            const long long p = pk + kk;
            sA[kk][i] = (i0 + i < M && p < p1) ? A[(long long)(i0 + i) * lda + p] : make_float2(0.f, 0.f);
        }
        if (NN) {
            for (int e = threadIdx.x; e < TN * TK; e += 256) {
                const int kk = e / TN, j = e % TN;
                const long long p = pk + kk;
                sB[kk][j] = (j0 + j < N && p < p1) ? B[p * ldb + j0 + j] : make_float2(0.f, 0.f);
            }
        } else {
            for (int e = threadIdx.x; e < TN * TK; e += 256) {
                const int j = e / TK, kk = e % TK;
                const long long p = pk + kk;
                float2 b = (j0 + j < N && p < p1) ? B[(long long)(j0 + j) * ldb + p] : make_float2(0.f, 0.f);
                b.y = -b.y;
                sB[kk][j] = b;
            }
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < TK; ++kk) {
            float2 a[4], b[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { a[u] = sA[kk][ty * 4 + u]; b[u] = sB[kk][tx * 4 + u]; }
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    acc[u][v].x = fmaf(a[u].x, b[v].x, acc[u][v].x); acc[u][v].x = fmaf(-a[u].y, b[v].y, acc[u][v].x);
                    acc[u][v].y = fmaf(a[u].x, b[v].y, acc[u][v].y); acc[u][v].y = fmaf(a[u].y, b[v].x, acc[u][v].y);
                }
        }
        __syncthreads();
        if (++since_flush == 32) {   // 512 terms per fp32 partial sum, then into fp64
            since_flush = 0;
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int v = 0; v < 4; ++v) {
                    dacc[u][v].x += acc[u][v].x; dacc[u][v].y += acc[u][v].y;
                    acc[u][v] = make_float2(0.f, 0.f);
                }
        }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            const int i = i0 + ty * 4 + u, j = j0 + tx * 4 + v;
            if (i < M && j < N)
                C[(long long)i * ldc + j] = make_float2((float)(dacc[u][v].x + acc[u][v].x), (float)(dacc[u][v].y + acc[u][v].y));
        }
}

// ---- Gram-Schmidt on row vectors Q[row][n] (ld entries apart) ---------------------------------------------------
// r[i] = <q_i, w> = sum_p conj(Q[i][p]) w[p], i < j: grid (j, splits); fp64 partial sums, double atomics
__global__ void __launch_bounds__(256) gs_dots_kernel(const float2* __restrict__ Q, long long ld, const float2* __restrict__ w,
                                                      long long n, double2* r) {
    const int i = blockIdx.x;
    const long long chunk = (n + gridDim.y - 1) / gridDim.y;
    const long long a = blockIdx.y * chunk, b = a + chunk < n ? a + chunk : n;
    const float2* q = Q + (long long)i * ld;
    double re = 0.0, im = 0.0;
    for (long long p = a + threadIdx.x; p < b; p += 256) {
        const float2 x = q[p], y = w[p];
        re += (double)x.x * y.x + (double)x.y * y.y;
        im += (double)x.x * y.y - (double)x.y * y.x;
    }
    for (int o = 16; o > 0; o >>= 1) { re += __shfl_xor_sync(0xffffffffu, re, o); im += __shfl_xor_sync(0xffffffffu, im, o); }
    __shared__ double sre[8], sim[8];
    if ((threadIdx.x & 31) == 0) { sre[threadIdx.x >> 5] = re; sim[threadIdx.x >> 5] = im; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int k = 1; k < 8; ++k) { re += sre[k]; im += sim[k]; }
        atomicAdd(&r[i].x, re); atomicAdd(&r[i].y, im);
    }
}

// w[p] -= sum_{i<j} r[i] Q[i][p]
__global__ void __launch_bounds__(256) gs_update_kernel(const float2* __restrict__ Q, long long ld, float2* __restrict__ w,
                                                        long long n, const double2* __restrict__ r, int j) {
    const long long p = blockIdx.x * 256ll + threadIdx.x;
    if (p >= n) return;
    float sx = 0.f, sy = 0.f;
    for (int i = 0; i < j; ++i) {
        const float2 q = Q[(long long)i * ld + p];
        const float rx = (float)r[i].x, ry = (float)r[i].y;
        sx = fmaf(rx, q.x, sx); sx = fmaf(-ry, q.y, sx);
        sy = fmaf(rx, q.y, sy); sy = fmaf(ry, q.x, sy);
    }
    float2 v = w[p];
    v.x -= sx; v.y -= sy;
    w[p] = v;
}

__global__ void __launch_bounds__(256) gs_norm_kernel(const float2* __restrict__ w, long long n, double* nrm2) {
    double s = 0.0;
    for (long long p = blockIdx.x * 256ll + threadIdx.x; p < n; p += (long long)gridDim.x * 256) {
        const float2 v = w[p];
        s += (double)v.x * v.x + (double)v.y * v.y;
    }
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(nrm2, s);
}

__global__ void __launch_bounds__(256) gs_scale_kernel(float2* __restrict__ w, long long n, const double* nrm2, float* out_norm) {
    const double nn = *nrm2;
    const float sc = nn > 0.0 ? (float)(1.0 / sqrt(nn)) : 0.f;
    if (out_norm != nullptr && blockIdx.x == 0 && threadIdx.x == 0) *out_norm = (float)sqrt(nn);
    for (long long p = blockIdx.x * 256ll + threadIdx.x; p < n; p += (long long)gridDim.x * 256) {
        float2 v = w[p];
        v.x *= sc; v.y *= sc;
        w[p] = v;
    }
}

// start vectors: counter-based hash -> uniform in [-1, 1)^2
__global__ void prep_random_kernel(float2* v, long long n, unsigned long long seed) {
    const long long i = blockIdx.x * 256ll + threadIdx.x;
    if (i >= n) return;
    unsigned long long x = (unsigned long long)i * 0x9E3779B97F4A7C15ull + seed;
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull; x ^= x >> 27; x *= 0x94D049BB133111EBull; x ^= x >> 31;
    v[i] = make_float2((float)(x & 0xffffff) / 8388608.f - 1.f, (float)((x >> 24) & 0xffffff) / 8388608.f - 1.f);
}

// zero the entries of every row outside the band [j_low, n_half)
__global__ void prep_band_kernel(float2* rows, long long bins, int nrows, int j_low, long long n_half) {
    const long long j = blockIdx.x * 256ll + threadIdx.x;
    if (j >= bins || (j >= j_low && j < n_half)) return;
    for (int r = 0; r < nrows; ++r) rows[(long long)r * bins + j] = make_float2(0.f, 0.f);
}

__global__ void prep_sigma_kernel(const float2* __restrict__ coeffs, float* __restrict__ sigma, int T, int k) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    double s = 0.0;
    for (int c = 0; c < k; ++c) { const float2 v = coeffs[(long long)t * k + c]; s += (double)v.x * v.x + (double)v.y * v.y; }
    sigma[t] = (float)sqrt(s);
}

template <bool NN>
cudaError_t cgemm(const float2* A, long long lda, const float2* B, long long ldb, float2* C, long long ldc, int M, int N,
                  long long p0, long long p1, cudaStream_t st) {
    const long long tiles = (long long)((N + TN - 1) / TN) * ((M + TM - 1) / TM);
    if (tiles < 1 || tiles > 0x7fffffffll) return cudaErrorInvalidConfiguration;
    cgemm_kernel<NN><<<(unsigned)tiles, 256, 0, st>>>(A, lda, B, ldb, C, ldc, M, N, p0, p1);
    return cudaGetLastError();
}

// Orthonormalise the rows of Q (nrows x n, ld apart) in place: classical Gram-Schmidt, each row projected twice.
// scratch: nrows double2 + 1 double.  norms (optional): the length of every row before its normalisation.
cudaError_t orthonormalise_rows(float2* Q, long long ld, long long n, int nrows, double2* r, double* nrm2, float* norms,
                                cudaStream_t st) {
    const int splits = (int)(n >= (1 << 16) ? 16 : (n >= 4096 ? 4 : 1));
    const unsigned gn = (unsigned)((n + 255) / 256);
    for (int j = 0; j < nrows; ++j) {
        float2* w = Q + (long long)j * ld;
        for (int pass = 0; pass < 2 && j > 0; ++pass) {
            cudaError_t e = cudaMemsetAsync(r, 0, (size_t)j * sizeof(double2), st);
            if (e != cudaSuccess) return e;
            gs_dots_kernel<<<dim3(j, splits), 256, 0, st>>>(Q, ld, w, n, r);
            gs_update_kernel<<<gn, 256, 0, st>>>(Q, ld, w, n, r, j);
            if ((e = cudaGetLastError()) != cudaSuccess) return e;
        }
        cudaError_t e = cudaMemsetAsync(nrm2, 0, sizeof(double), st);
        if (e != cudaSuccess) return e;
        gs_norm_kernel<<<gn < 1024 ? gn : 1024, 256, 0, st>>>(w, n, nrm2);
        gs_scale_kernel<<<gn < 1024 ? gn : 1024, 256, 0, st>>>(w, n, nrm2, norms ? norms + j : nullptr);
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
    return cudaSuccess;
}

}  // namespace

// Bytes of the float2 part of the workspace (G, Va, Vb), rounded up to 16: the Gram-Schmidt scratch behind it is read
// as double2 (128-bit loads), and S (S + 2k) float2 entries are 8 mod 16 bytes when the number of templates S is odd.
static size_t prep_vectors_bytes(int S, int k) {
    return (((size_t)S * S + 2ull * k * S) * sizeof(float2) + 15) & ~(size_t)15;
}

size_t prep_basis_workspace_bytes(int S, int k) {
    // G (S x S) + two sets of k row vectors of length S + Gram-Schmidt scratch
    return prep_vectors_bytes(S, k) + (size_t)k * sizeof(double2) + 1024;
}

// templates: S x bins (rows), band [j_low, n_half); basis_out: k x bins.  eig_out (optional): k floats, the lengths
// ||C v_i|| of the last iteration (estimates of the leading eigenvalues of C = squared singular values of T).
cudaError_t launch_prep_basis(const float2* templates, int S, long long bins, int j_low, long long n_half, int k,
                              int iterations, unsigned long long seed, void* workspace, float2* basis_out,
                              float* eig_out, cudaStream_t st) {
    float2* G = reinterpret_cast<float2*>(workspace);
    float2* Va = G + (size_t)S * S;       // k x S: rows = conj of the iteration vectors (V^H)
    float2* Vb = Va + (size_t)k * S;
    double2* r = reinterpret_cast<double2*>(reinterpret_cast<char*>(workspace) + prep_vectors_bytes(S, k));
    double* nrm2 = reinterpret_cast<double*>(r + k);
    cudaError_t e;
    // C = T T^H over the band
    if ((e = cgemm<false>(templates, bins, templates, bins, G, S, S, S, j_low, n_half, st)) != cudaSuccess) return e;
    prep_random_kernel<<<(unsigned)(((long long)k * S + 255) / 256), 256, 0, st>>>(Va, (long long)k * S, seed);
    if ((e = orthonormalise_rows(Va, S, S, k, r, nrm2, nullptr, st)) != cudaSuccess) return e;
    for (int it = 0; it < iterations; ++it) {
        // rows of Va are v_i^H; (C v_i)^H = v_i^H C (C Hermitian): Vb = Va C, i.e. Vb[i][s] = sum_p Va[i][p] C[p][s]
        if ((e = cgemm<true>(Va, S, G, S, Vb, S, k, S, 0, S, st)) != cudaSuccess) return e;
        if ((e = orthonormalise_rows(Vb, S, S, k, r, nrm2, it == iterations - 1 ? eig_out : nullptr, st)) != cudaSuccess) return e;
        float2* t = Va; Va = Vb; Vb = t;
    }
    // P = orth(V^H T): basis[i][j] = sum_s Va[i][s] T[s][j]
    if ((e = cgemm<true>(Va, S, templates, bins, basis_out, bins, k, (int)bins, 0, S, st)) != cudaSuccess) return e;
    prep_band_kernel<<<(unsigned)((bins + 255) / 256), 256, 0, st>>>(basis_out, bins, k, j_low, n_half);
    return orthonormalise_rows(basis_out, bins, bins, k, r, nrm2, nullptr, st);
}

// D = T P^H over the band, sigma_t = ||c_t||_2
cudaError_t launch_prep_coeffs_from_templates(const float2* templates, int T, const float2* basis, int k, long long bins,
                                              int j_low, long long n_half, float2* coeffs_out, float* sigma_out,
                                              cudaStream_t st) {
    cudaError_t e = cgemm<false>(templates, bins, basis, bins, coeffs_out, k, T, k, j_low, n_half, st);
    if (e != cudaSuccess) return e;
    if (sigma_out != nullptr) prep_sigma_kernel<<<(T + 255) / 256, 256, 0, st>>>(coeffs_out, sigma_out, T, k);
    return cudaGetLastError();
}

}  // namespace rbmf
