// Internal declarations shared by the translation units of librbmf.so (not part of the C ABI).
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "rbmf.h"

namespace rbmf {

constexpr int kFftKC = 8;          // basis columns per FFT CTA (64-byte row segments)
constexpr int kGemmBM = 128;       // time bins per GEMM tile (UMMA M)
constexpr int kGemmTT = 128;       // templates per GEMM tile (UMMA N = 2*kGemmTT: re | im rows)
constexpr int kGemmBK = 64;        // bf16 elements per K block (= one 128-byte swizzle row)

// Device views handed to the FFT kernels.
struct FftArgs {
    const float2* in;        // pass 1: basisT (rows j < N/2, k columns); pass 2: Y
    const float2* strain;    // pass 1: scaled strain ds[j] (main) or dS[j] = ds[j] S(j) (fold)
    float2* out;             // pass 1: Y; pass 2: beta (may be null)
    uint16_t* plane_hi;      // pass 2 plane modes: (rows) x 2k bf16
    uint16_t* plane_lo;
    const float2* tw_L;      // e^{2 pi i m / L}, m < L (table of this pass's length)
    const float2* tw_lo;     // e^{2 pi i m / Ntot}, m < 1024
    const float2* tw_hi;     // e^{2 pi i 1024 m / Ntot}, m < max(1, Ntot/1024)
    int k;                   // columns
    int lines;               // O = Ntot / L: number of independent lines (grid.x)
    int j_low;               // first in-band bin
    int n_half;              // N/2 (first out-of-band bin)
    int fold;                // pass 1 fold mode: number of aliases to sum = max(1, w/2); else 1
    int fold_stride;         // M = N/w (bins between aliases)
};

struct GemmArgs {
    rbmf_candidate* cand;
    unsigned long long* counters;   // [0] = candidates, [1] = triggers
    unsigned long long cand_cap;
    float thr1_sq;
    int T;                    // real templates (rows >= T are padding)
    int M;                    // time bins N/w
    int k2;                   // 2k (reals along K)
    int num_tb;               // template blocks  = Tpad / 128
    int num_ib;               // time-bin blocks  = M / 128
    int group;                // template blocks per raster group
};

struct Stage2Args {
    const rbmf_candidate* cand;
    const float2* cs;         // T x k: conj(c_tk) / sigma_t
    const float2* beta;       // N x k
    rbmf_trigger* out;
    unsigned long long* counters;
    unsigned long long cand_cap;
    unsigned long long trig_cap;
    float thr2_sq;
    int k;
    int w;
};

// ---- launchers (each returns the cudaError_t of the launch) -------------------------------------
cudaError_t launch_init_tables(float2* tw_L_all, float2* tw_lo_main, float2* tw_hi_main, float2* tw_lo_avg,
                               float2* tw_hi_avg, float2* S_table, int64_t N, int64_t M, int w, cudaStream_t st);
cudaError_t launch_transpose_basis(const float2* basis, float2* basisT, int k, int64_t bins, int j_low,
                                   int n_half, cudaStream_t st);
cudaError_t launch_prep_coeffs(const float2* coeffs, const float* sigma, float2* cs, uint16_t* c_hi,
                               uint16_t* c_lo, int T, int Tpad, int k, cudaStream_t st);
cudaError_t launch_prep_strain(const float2* strain, const float2* S_table, float2* ds, float2* dS,
                               int n_half, float scale, cudaStream_t st);
cudaError_t launch_fft_pass1(const FftArgs& a, int logL, bool fold, cudaStream_t st);
// mode: 0 = write beta, 1 = write planes, 2 = both
cudaError_t launch_fft_pass2(const FftArgs& a, int logL, int mode, cudaStream_t st);
cudaError_t launch_gemm_simt(const uint16_t* a_hi, const uint16_t* a_lo, const uint16_t* c_hi,
                             const uint16_t* c_lo, const GemmArgs& g, cudaStream_t st);
cudaError_t launch_gemm_tcgen05(const CUtensorMap& tmA_hi, const CUtensorMap& tmA_lo, const CUtensorMap& tmB_hi,
                                const CUtensorMap& tmB_lo, const GemmArgs& g, int num_sms, cudaStream_t st);
cudaError_t gemm_tcgen05_configure();   // sets the dynamic shared memory attribute once
cudaError_t launch_stage2(const Stage2Args& a, int num_sms, cudaStream_t st);

// Offset (in float2 entries) of the length-2^logL twiddle table inside tw_L_all; tables for logL = 5..10.
__host__ __device__ inline int tw_table_offset(int logL) { return (1 << logL) - 32; }
constexpr int kTwAllEntries = 2048 - 32;

}  // namespace rbmf
