// The paper's two template-route filters as on-GPU comparators of the basis/GEMM route:
//
//   flat template method (Eq. 13 :238, the 100 ms cuFFT baseline of :338): one full-length inverse FFT
//     per template, rho_t[n] = (s / sigma_t) sum_j d[j] conj(h_t[j]) e^{2 pi i j n / N}, every sample thresholded;
//   fast first stage by templates (Eq. 10-12; cost Eq. 14 :244): the averaged series straight from
//     an alias-folded spectrum and a SHORT inverse FFT,
//         Omega_t(f') = sum_l G_t[l M + f'] S(l M + f'),  M = N / w,  G_t = s d conj(h_t) / sigma_t,
//         S(f) = (1/w) sum_{r<w} e^{2 pi i f r / N},      rho_bar_t[b] = sum_{f' < M} Omega_t(f') e^{2 pi i f' b / M}
//     (Eq. 12 as printed is garbled; this is reading R14 of DESIGN.md, pinned in tests/test_oracle_pins.py).
//
// Both reuse kernel 1 (fft_tma.cu) unchanged, with TEMPLATES in the place of basis vectors, a slab of columns at a time:
// the flat method lays a slab of templates out in the order pass 1 reads (layout kernel of prep_kernels.cu) and runs
// the length-N transform; the fast first stage folds the slab into Omega (fold kernel below), hands conj(Omega) to a
// length-2M transform as a one-sided spectrum (unit "strain"), and keeps the even outputs: out[2b] =
// sum_{f'<M} Omega(f') e^{2 pi i f' 2b / 2M} = rho_bar[b].  A scan kernel thresholds the transform's output and appends
// triggers (flat) or first-stage candidates + the per-bin histogram stage 2 needs (fast first stage).
#include "rbmf_internal.h"

namespace rbmf {

namespace {

// S[j] = (1/w) sum_{r<w} e^{2 pi i j r / N}, j < N/2, in fp64 (Eq. 11)
__global__ void tm_s_table_kernel(float2* S, long long N, int w) {
    const long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (j >= N / 2) return;
    double re = 0.0, im = 0.0;
    for (int r = 0; r < w; ++r) {
        double s, c;
        sincospi(2.0 * (double)((j * r) % N) / (double)N, &s, &c);
        re += c; im += s;
    }
    S[j] = make_float2((float)(re / w), (float)(im / w));
}

__global__ void tm_fill_ones_kernel(float2* p, long long n) {
    const long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (i < n) p[i] = make_float2(1.f, 0.f);
}

// inv_sigma[t] = 1 / sigma_t (0 disables a template whose sigma is not a positive finite number); NULL sigma => 1
__global__ void tm_inv_sigma_kernel(const float* sigma, float* inv_sigma, int T) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= T) return;
    float v = 1.f;
    if (sigma != nullptr) {
        const float sg = sigma[t];
        v = (sg > 0.f && sg <= 3.0e38f) ? 1.0f / sg : 0.f;
    }
    inv_sigma[t] = v;
}

// Fold of Eq. 10-12 for the templates t0 .. t0 + 4 gridDim.z of the bank, written as conj(Omega) in the pass-1 order
// of the length-2M transform: out[chunk][tile][j1 < L1/2][line < sub][C], f' = j1 L2 + (tile sub + line) < M.
// Block = 32 f'-columns (j2) x 32 rows (j1) x one chunk of 4 templates, transposed through shared memory so that both
// the reads (consecutive j of one template) and the writes (consecutive j1 of one line) are coalesced.
__global__ void tm_fold_kernel(const float2* __restrict__ templates, const float2* __restrict__ strain,
                               const float2* __restrict__ S, float2* __restrict__ out, long long bins, int j_low,
                               long long n_half, int w, float scale, int t0, int T, int logL1, int logL2, int sub) {
    __shared__ float2 tile[kFftC][32][33];
    const int L2 = 1 << logL2, H = (1 << logL1) / 2;
    const long long M = (long long)H * L2;   // bins of the short transform's one-sided input = N / w
    const int chunk = blockIdx.z;
    const int j2_0 = blockIdx.x * 32, j1_0 = blockIdx.y * 32;
    const int tx = threadIdx.x % 32, ty = threadIdx.x / 32;   // 32 x 8
    const int nl = w / 2 > 0 ? w / 2 : 1;    // G vanishes for j >= N/2: only l < w/2 contribute (w = 1: l = 0)
    for (int c = 0; c < kFftC; ++c) {
        const int t = t0 + chunk * kFftC + c;
        for (int r = ty; r < 32; r += 8) {
            const int j1 = j1_0 + r, j2 = j2_0 + tx;
            float2 acc = make_float2(0.f, 0.f);
            if (j1 < H && j2 < L2 && t < T) {
                const long long fp = (long long)j1 * L2 + j2;
                for (int l = 0; l < nl; ++l) {
                    const long long j = (long long)l * M + fp;
                    if (j >= j_low && j < n_half) {
                        const float2 d = strain[j], h = templates[(long long)t * bins + j], s = S[j];
                        const float2 g = make_float2(d.x * h.x + d.y * h.y, d.y * h.x - d.x * h.y);   // d conj(h)
                        acc.x += g.x * s.x - g.y * s.y;
                        acc.y += g.x * s.y + g.y * s.x;
                    }
                }
            }
            tile[c][r][tx] = make_float2(acc.x * scale, -acc.y * scale);   // conj(Omega): pass 1 multiplies by conj again
        }
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int j2 = j2_0 + r;
        if (j2 >= L2) continue;
        for (int e = tx; e < 32 * kFftC; e += 32) {
            const int j1 = j1_0 + e / kFftC, c = e % kFftC;
            if (j1 < H)
                out[((((size_t)chunk * (L2 / sub) + j2 / sub) * fft_p1_rows(logL1) + fft_p1_row(logL1, j1)) * sub +
                     j2 % sub) * kFftC + c] = tile[c][e / kFftC][r];
        }
    }
}

// Threshold scan of a transform's output beta[chunk][n][C]: rows n = step * i, i < nout; column c of chunk ch is
// template t0 + 4 ch + c.  Appends {template, i, value / sigma} records where |value / sigma|^2 >= thr_sq (one
// list-space reservation per warp); with bin_count != NULL also counts the entries written per i (first-stage mode).
__global__ void __launch_bounds__(256) tm_scan_kernel(const float2* __restrict__ beta, long long Nrows, int step,
                                                      int nout, const float* __restrict__ inv_sigma, int t0, int T,
                                                      float thr_sq, rbmf_trigger* __restrict__ out,
                                                      unsigned long long* counter, unsigned long long cap,
                                                      unsigned* bin_count) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int ch = blockIdx.y, lane = threadIdx.x & 31;
    float2 v[kFftC];
    unsigned mask = 0;
    if (i < nout) {
        const float4* p = reinterpret_cast<const float4*>(beta + ((size_t)ch * Nrows + (size_t)i * step) * kFftC);
        const float4 a = __ldg(p), b = __ldg(p + 1);
        v[0] = make_float2(a.x, a.y); v[1] = make_float2(a.z, a.w);
        v[2] = make_float2(b.x, b.y); v[3] = make_float2(b.z, b.w);
#pragma unroll
        for (int c = 0; c < kFftC; ++c) {
            const int t = t0 + ch * kFftC + c;
            const float is = t < T ? __ldg(inv_sigma + t) : 0.f;
            v[c].x *= is; v[c].y *= is;
            if (t < T && is > 0.f && !(v[c].x * v[c].x + v[c].y * v[c].y < thr_sq)) mask |= 1u << c;
        }
    }
    const int cnt = __popc(mask);
    if (__ballot_sync(0xffffffffu, cnt != 0) == 0) return;
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int x = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += x;
    }
    const int total = __shfl_sync(0xffffffffu, incl, 31);
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(counter, (unsigned long long)total);
    base = __shfl_sync(0xffffffffu, base, 0);
    unsigned long long idx = base + (unsigned long long)(incl - cnt);
    int written = 0;
#pragma unroll
    for (int c = 0; c < kFftC; ++c) {
        if ((mask >> c) & 1u) {
            if (idx < cap) {
                rbmf_trigger r;
                r.template_id = t0 + ch * kFftC + c; r.time_index = i; r.snr_re = v[c].x; r.snr_im = v[c].y;
                out[idx] = r;
                ++written;
            }
            ++idx;
        }
    }
    if (bin_count != nullptr && written > 0) atomicAdd(bin_count + i, (unsigned)written);
}

}  // namespace

cudaError_t launch_tm_tables(float2* S, float2* ones, long long N, int w, long long n_ones, cudaStream_t st) {
    tm_s_table_kernel<<<(unsigned)((N / 2 + 255) / 256), 256, 0, st>>>(S, N, w);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    tm_fill_ones_kernel<<<(unsigned)((n_ones + 255) / 256), 256, 0, st>>>(ones, n_ones);
    return cudaGetLastError();
}

cudaError_t launch_tm_inv_sigma(const float* sigma, float* inv_sigma, int T, cudaStream_t st) {
    tm_inv_sigma_kernel<<<(T + 255) / 256, 256, 0, st>>>(sigma, inv_sigma, T);
    return cudaGetLastError();
}

cudaError_t launch_tm_fold(const float2* templates, const float2* strain, const float2* S, float2* out, long long bins,
                           int j_low, long long n_half, int w, float scale, int t0, int T, int ncols, int logL1,
                           int logL2, int sub, cudaStream_t st) {
    const int L2 = 1 << logL2, H = (1 << logL1) / 2;
    dim3 grid((unsigned)((L2 + 31) / 32), (unsigned)((H + 31) / 32), (unsigned)(ncols / kFftC));
    tm_fold_kernel<<<grid, 256, 0, st>>>(templates, strain, S, out, bins, j_low, n_half, w, scale, t0, T, logL1, logL2,
                                         sub);
    return cudaGetLastError();
}

cudaError_t launch_tm_scan(const float2* beta, long long Nrows, int step, int nout, const float* inv_sigma, int t0,
                           int T, int ncols, float thr_sq, rbmf_trigger* out, unsigned long long* counter,
                           unsigned long long cap, unsigned* bin_count, cudaStream_t st) {
    dim3 grid((unsigned)((nout + 255) / 256), (unsigned)(ncols / kFftC));
    tm_scan_kernel<<<grid, 256, 0, st>>>(beta, Nrows, step, nout, inv_sigma, t0, T, thr_sq, out, counter, cap, bin_count);
    return cudaGetLastError();
}

}  // namespace rbmf
