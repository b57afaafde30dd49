// Internal declarations shared by the translation units of librbmf.so (not part of the C ABI).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "rbmf.h"

namespace rbmf {

constexpr int kFftC = 4;           // basis columns per FFT chunk (32-byte row segments)
constexpr int kFftThreads = 256;   // threads per FFT consumer group
constexpr int kMaxChunks = 256;    // k <= 1024
constexpr int kGemmBM = 128;       // time bins per GEMM tile (UMMA M)
constexpr int kGemmTT = 128;       // templates per GEMM tile (UMMA N = 2*kGemmTT: re | im rows)
constexpr int kGemmBK = 64;        // bf16 elements per K block (= one 128-byte swizzle row = 32 basis columns)

// Per-length configuration of the in-CTA transform: L = R0 * R1, two Stockham stages.
// A thread owns one column and R0 elements; W = L / R0 = R1 threads cooperate on one column of one line.
__host__ __device__ constexpr int fft_r0(int logL) { return logL >= 9 ? 32 : (logL >= 7 ? 16 : 8); }
__host__ __device__ constexpr int fft_r1(int logL) { return (1 << logL) / fft_r0(logL); }
// lines (independent transforms) a 256-thread consumer group works on in lockstep = lines per tile
__host__ __device__ constexpr int fft_sub(int logL) { return kFftThreads / (fft_r1(logL) * kFftC); }

// Input of a pass-1 tile (sub lines j2 of one chunk), laid out in global memory exactly as it sits in the tile buffer, so
// that the producer moves it with TWO bulk copies (a bulk copy costs the producer warp ~150 cycles to issue; sixteen
// 2 KB pieces into padded rows made the producer, not the consumers, the kernel's bottleneck):
//   basis part  [row(j1)][line][C], j1 < L1/2, with one pad row after every 32 rows when a row is 64 bytes
//               (L1 = 1024: keeps stage 1's shared-memory reads conflict-free, see fft_tma.cu);
//   strain part [line][L1/2 + spad] entries (lines offset so that the lines a warp reads fall into different banks).
__host__ __device__ constexpr bool fft_p1_pad(int logL) { return fft_sub(logL) * kFftC * 8 == 64; }
__host__ __device__ constexpr int fft_p1_rows(int logL) {
    return fft_p1_pad(logL) ? (1 << logL) / 2 + (1 << logL) / 64 : (1 << logL) / 2;
}
__host__ __device__ constexpr int fft_p1_row(int logL, int j1) { return fft_p1_pad(logL) ? j1 + (j1 >> 5) : j1; }
__host__ __device__ constexpr int fft_spad(int logL) { return 16 / fft_sub(logL) > 2 ? 16 / fft_sub(logL) : 2; }
__host__ __device__ constexpr int fft_strain_row(int logL) { return (1 << logL) / 2 + fft_spad(logL); }

// Scheduler words (uint32) in the workspace: [0] ticket, [16 + v] pass-1 tiles done of virtual chunk v = c * nb + b
// (c = chunk of 4 basis columns, b = segment of the batch): 16 + kMaxChunks * max_batch words.
constexpr int kSchedBase = 16;
// Counter block (uint64 words) at the head of the scheduler area, zeroed by every rbmf_filter:
//   [0] stage-1 list entries requested by kernel 2, [1] triggers, [2] confirmed candidates (screen mode),
//   [3] cursor of the by-bin candidate array, [4] stage-2 work items, [5] stage-2 ticket, [8] rbmf_filter_host's count.
constexpr int kCounterBytes = 128;
constexpr int kEvRing = 64;         // timed calls whose stage events a plan keeps (rbmf_get_stage_ms_history)
constexpr int kStage2Chunk = 128;   // candidates per stage-2 work item (one CTA of 4 warps)

// Device views handed to the fused FFT kernel.
struct FftArgs {
    const float2* basisP;    // [chunk][tile][fft_p1_row(j1)][line][C], j2 = tile * sub + line: conj NOT applied, zero outside the band
    const float2* dsT;       // [segment][j2 < L2][fft_strain_row]: s * d[j1 L2 + j2] at entry j1 < L1/2
    const float2* tw1_a;     // pass 1 stage-1 twiddles  [q < R1][b < R0] = e^{2 pi i q b / L1}
    const float2* tw1_b;     // pass 2 stage-1 twiddles, same for L2
    const float2* twN;       // inter-pass twiddles as two factor tables, [j2][b < R0] then [j2][m < R1] (prep_kernels.cu)
    float2* beta;            // [chunk][n < N][C]; between the passes it holds Y[n1][j2] at index n1 + L1 j2
    uint16_t* plane_hi;      // [kb = col / 32][bin < M][64]: bf16 (re, im) of column col % 32
    uint16_t* plane_lo;
    unsigned* sched;         // kSchedBase + nchunk * nb words
    long long N;
    int M;                   // rows of the planes = max_batch * N / w
    int nchunk;              // k / C
    int w;
    float inv_w;
    int lookahead;           // (virtual) chunks pass 1 runs ahead of pass 2 in the work queue (their Y must fit in L2)
    int nb;                  // segments of the batch: virtual chunk v = c * nb + b reads basis chunk c, strain b
    int seg_major;           // 1: v = b * nchunk + c instead (every segment streams the basis from HBM again)
    int Mseg;                // bins per segment (N / w); segment b's bins are [b Mseg, (b + 1) Mseg) of the planes
    int plane_fp16;          // 1: write ONE fp16 plane (screen mode) into plane_hi; 0: bf16 hi + lo planes
    int no_planes;           // 1: skip step a3's plane output altogether (template routes read beta directly)
};

struct GemmArgs {
    // screen mode only (see gemm_tcgen05.cu): per-bin norms, per-template-block norm maxima, bound constants
    const float* bin_norm;    // M floats: upper bound of ||beta^avg[i]||_2
    const float* tnorm_blk;   // num_tb floats: max_t ||c_t||_2 / sigma_t over the block's templates
    float thr1;
    float kappa1, kappa2, slack;
    rbmf_candidate* cand;
    unsigned* bin_count;            // per (segment, bin): entries written to `cand` (histogram for stage 2's grouping)
    unsigned long long* counters;   // [0] = candidates, [1] = triggers
    unsigned long long cand_cap;
    float thr1_sq;
    int T;                    // real templates (rows >= T are padding)
    int M;                    // time bins of the whole batch, nb * N / w
    int k2;                   // 2k (reals along K)
    int num_tb;               // template blocks  = Tpad / 128
    int num_ib;               // time-bin blocks  = M / 128
    int group;                // template blocks per raster group
};

struct Stage2Args {
    const rbmf_candidate* cand;
    // by-bin path: candidates regrouped by bin (bin_count from kernel 2; alloc -> bin_start + items; scatter -> sorted)
    unsigned* bin_count;
    unsigned* bin_start;
    int4* items;                 // {bin, first entry in `sorted`, entries (<= kStage2Chunk), 0}
    rbmf_candidate* sorted;
    int Mseg;                    // bins per segment (N / w); bin / Mseg = segment of the batch
    int Mtot;                    // nb * Mseg
    size_t seg_stride;           // float2 entries between the beta arrays of consecutive segments
    int smem_bytes;              // dynamic shared memory of the score kernel (beta block of one bin)
    const float2* cs;         // T x k: conj(c_tk) / sigma_t
    const float2* beta;       // [chunk][n][C]
    rbmf_trigger* out;
    unsigned long long* trig_counter;   // list position counter of `out`: counters + 1, or a counter shared by the
                                        // plans of a bank set (then counters[1] still counts this plan's own triggers)
    int template_offset;                // added to the template id of every trigger (sub-bank base in a bank set)
    rbmf_candidate* confirmed;   // screen mode: candidates whose fp32 averaged SNR passes thr1 (counters[2])
    float thr1_sq;
    int screen;                  // 1: `cand` is the screened superset; confirm before scoring
    unsigned long long* counters;
    unsigned long long cand_cap;
    unsigned long long trig_cap;
    long long N;
    float thr2_sq;
    int k;
    int w;
};

// ---- launchers (each returns the cudaError_t of the launch) -------------------------------------
cudaError_t launch_init_tables(float2* tw1_a, float2* tw1_b, float2* twN, int logL1, int logL2, cudaStream_t st);
cudaError_t launch_layout_basis(const float2* basis, float2* basisP, int k, int64_t bins, int j_low, int logL1,
                                int logL2, int sub, int rows_valid, cudaStream_t st);
// template routes (template_route.cu)
cudaError_t launch_tm_tables(float2* S, float2* ones, long long N, int w, long long n_ones, cudaStream_t st);
cudaError_t launch_tm_inv_sigma(const float* sigma, float* inv_sigma, int T, cudaStream_t st);
cudaError_t launch_tm_fold(const float2* templates, const float2* strain, const float2* S, float2* out, long long bins,
                           int j_low, long long n_half, int w, float scale, int t0, int T, int ncols, int logL1,
                           int logL2, int sub, cudaStream_t st);
cudaError_t launch_tm_scan(const float2* beta, long long Nrows, int step, int nout, const float* inv_sigma, int t0,
                           int T, int ncols, float thr_sq, rbmf_trigger* out, unsigned long long* counter,
                           unsigned long long cap, unsigned* bin_count, cudaStream_t st);
cudaError_t launch_prep_coeffs(const float2* coeffs, const float* sigma, float2* cs, uint16_t* c_hi,
                               uint16_t* c_lo, uint16_t* c_h16, float* tnorm_blk, int T, int Tpad, int k,
                               cudaStream_t st);
cudaError_t launch_bin_norm(const uint16_t* plane_h16, float* bin_norm, int M, int Mplane, int nkb, cudaStream_t st);
cudaError_t launch_prep_strain(const float2* strain, float2* dsT, int logL1, int logL2, float scale, int nb,
                               cudaStream_t st);
// Fused FFT (a1-a3): configure once per (logL1, logL2); then launch with one CTA per SM.  tmY: 3-D fp32 tensor map
// over the beta array, dims {2 C L1, L2, k/C}, box {2 C sub2, min(L2, 256), 1} (the Y rows of a pass-2 tile).
cudaError_t fft_tma_configure(int logL1, int logL2, size_t* smem_bytes);
cudaError_t launch_fft_tma(const CUtensorMap& tmY, const FftArgs& a, int logL1, int logL2, int grid, cudaStream_t st);
cudaError_t launch_gemm_simt(const uint16_t* a_hi, const uint16_t* a_lo, const uint16_t* c_hi,
                             const uint16_t* c_lo, const GemmArgs& g, int Mplane, cudaStream_t st);
cudaError_t launch_gemm_tcgen05(const CUtensorMap& tmA_hi, const CUtensorMap& tmA_lo, const CUtensorMap& tmB_hi,
                                const CUtensorMap& tmB_lo, const GemmArgs& g, int num_sms, cudaStream_t st);
// screen mode: one fp16 product; tmA = beta^avg fp16 plane, tmB = coefficient fp16 plane
// (pair_clusters > 0: the 2-CTA cluster kernel, which multicasts the coefficient tile and needs tmB_half, the same
// plane with a 128-row box)
cudaError_t launch_gemm_screen(const CUtensorMap& tmA, const CUtensorMap& tmB, const CUtensorMap& tmB_half,
                               int pair_clusters, const GemmArgs& g, int num_sms, cudaStream_t st);
cudaError_t gemm_screen_pair_clusters(int num_sms, int* clusters);
cudaError_t gemm_tcgen05_configure();   // sets the dynamic shared memory attribute once
cudaError_t launch_stage2(const Stage2Args& a, int num_sms, cudaStream_t st);          // one warp per candidate
cudaError_t launch_stage2_bybin(const Stage2Args& a, int num_sms, cudaStream_t st);    // regrouped by bin (default)
int stage2_bybin_smem(int w, int k);
// preparation (prep_basis.cu): PCA of a (sub-)bank and projection of templates onto a basis
size_t prep_basis_workspace_bytes(int S, int k);
cudaError_t launch_prep_basis(const float2* templates, int S, long long bins, int j_low, long long n_half, int k,
                              int iterations, unsigned long long seed, void* workspace, float2* basis_out,
                              float* eig_out, cudaStream_t st);
cudaError_t launch_prep_coeffs_from_templates(const float2* templates, int T, const float2* basis, int k, long long bins,
                                              int j_low, long long n_half, float2* coeffs_out, float* sigma_out,
                                              cudaStream_t st);
// front end (fft_r2c.cu): forward real-to-complex FFT of nb series of N = 2^logN samples + whitening
cudaError_t r2c_configure();
cudaError_t launch_r2c_table(float2* twF, long long N, cudaStream_t st);
cudaError_t launch_r2c(const float* x, const float* inv_asd, float2* S, float2* Z, float2* out, const float2* twF,
                       int logN, int nb, cudaStream_t st);   // shared memory of the by-bin score kernel; 0 = does not fit

}  // namespace rbmf
