// The step in front of the path: time-domain strain -> forward real-to-complex FFT -> whitening.
//   d[j] = inv_asd[j] * sum_n x[n] e^{-2 pi i j n / N},  j = 0 .. N/2        (PAPER.md:175 step 1, :177 "divided by
//   sqrt(S_n)"; the unnormalised forward DFT of SURVEY.md App. A)
// One real series of N samples is 4 MB at N = 2^20 -- three orders of magnitude less than the basis the path streams
// per segment -- so this is a plain, exact-twiddle implementation, not a tuned one:
//   z[m] = x[2m] + i x[2m+1], m < Nh = N/2 (the real array read as float2);
//   Z = forward complex DFT of z by the four-step split Nh = A B (n = a B + b, j = c + A d):
//       pass 1 (per b): length-A transform over a, times e^{-2 pi i b c / Nh}  -> S[c][b]
//       pass 2 (per c): length-B transform over b                             -> Z[c + A d]
//     each pass a radix-2 decimation-in-time transform in shared memory (bit-reversed load, log2 L in-place stages);
//   d[j] = E + e^{-2 pi i j / N} O,  E = (Z[j] + conj Z[Nh - j]) / 2,  O = -i (Z[j] - conj Z[Nh - j]) / 2.
// All twiddles come from one table twF[m] = e^{-2 pi i m / N}, m < N/2, evaluated in fp64 (sincospi).
#include <mutex>

#include "rbmf_internal.h"

namespace rbmf {

namespace {

constexpr int TL = 8;   // lines per CTA

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

__global__ void r2c_table_kernel(float2* twF, long long N) {
    const long long m = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (m >= N / 2) return;
    double s, c;
    sincospi(-2.0 * (double)m / (double)N, &s, &c);
    twF[m] = make_float2((float)c, (float)s);
}

// In-place radix-2 DIT stages on sm[pos * stride_pos + line * stride_line], pos < L (already bit-reversed), TL lines.
// Stage s pairs (i, i + 2^s) with e^{-2 pi i q / 2^(s+1)} = twF[q 2^(logN - 1 - s)], q = i mod 2^s.
__device__ __forceinline__ void dit_stages(float2* sm, int logL, int stride_pos, int stride_line, const float2* twF,
                                           int logN) {
    const int L = 1 << logL;
    for (int s = 0; s < logL; ++s) {
        const int half = 1 << s;
        for (int e = threadIdx.x; e < (L / 2) * TL; e += blockDim.x) {
            const int p = e / TL, ln = e % TL;
            const int q = p & (half - 1);
            const int i = ((p >> s) << (s + 1)) + q;
            const float2 w = __ldg(twF + ((size_t)q << (logN - 1 - s)));
            float2* lo = sm + i * stride_pos + ln * stride_line;
            float2* hi = sm + (i + half) * stride_pos + ln * stride_line;
            const float2 u = *lo, v = cmulf(*hi, w);
            *lo = make_float2(u.x + v.x, u.y + v.y);
            *hi = make_float2(u.x - v.x, u.y - v.y);
        }
        __syncthreads();
    }
}

// pass 1: CTA = TL consecutive b of segment blockIdx.y
__global__ void __launch_bounds__(256) r2c_pass1_kernel(const float2* __restrict__ z_all, float2* __restrict__ S_all,
                                                        const float2* __restrict__ twF, int logA, int logB, int logN) {
    extern __shared__ float2 sm[];   // [A][TL]
    const int A = 1 << logA, B = 1 << logB;
    const size_t Nh = (size_t)A * B;
    const float2* z = z_all + (size_t)blockIdx.y * Nh;
    float2* S = S_all + (size_t)blockIdx.y * Nh;
    const int b0 = blockIdx.x * TL;
    for (int e = threadIdx.x; e < A * TL; e += blockDim.x) {
        const int a = e / TL, ln = e % TL;
        const int ar = (int)(__brev((unsigned)a) >> (32 - logA));
        sm[ar * TL + ln] = z[(size_t)a * B + b0 + ln];
    }
    __syncthreads();
    dit_stages(sm, logA, TL, 1, twF, logN);
    for (int e = threadIdx.x; e < A * TL; e += blockDim.x) {
        const int c = e / TL, ln = e % TL;
        const size_t m = 2 * (size_t)(b0 + ln) * c;   // e^{-2 pi i b c / Nh} = e^{-2 pi i (2 b c) / N}, 2 b c < N
        float2 w = m < Nh ? __ldg(twF + m) : __ldg(twF + (m - Nh));
        if (m >= Nh) w = make_float2(-w.x, -w.y);
        S[(size_t)c * B + b0 + ln] = cmulf(sm[c * TL + ln], w);
    }
}

// pass 2: CTA = TL consecutive c of segment blockIdx.y
__global__ void __launch_bounds__(256) r2c_pass2_kernel(const float2* __restrict__ S_all, float2* __restrict__ Z_all,
                                                        const float2* __restrict__ twF, int logA, int logB, int logN) {
    extern __shared__ float2 sm[];   // [B][TL]
    const int A = 1 << logA, B = 1 << logB;
    const size_t Nh = (size_t)A * B;
    const float2* S = S_all + (size_t)blockIdx.y * Nh;
    float2* Z = Z_all + (size_t)blockIdx.y * Nh;
    const int c0 = blockIdx.x * TL;
    for (int e = threadIdx.x; e < B * TL; e += blockDim.x) {
        const int ln = e / B, b = e % B;   // rows of S are contiguous in b
        const int br = (int)(__brev((unsigned)b) >> (32 - logB));
        sm[br * TL + ln] = S[(size_t)(c0 + ln) * B + b];
    }
    __syncthreads();
    dit_stages(sm, logB, TL, 1, twF, logN);
    for (int e = threadIdx.x; e < B * TL; e += blockDim.x) {
        const int d = e / TL, ln = e % TL;
        Z[(size_t)(c0 + ln) + (size_t)A * d] = sm[d * TL + ln];
    }
}

// split of the packed transform + whitening; one thread per output bin j = 0 .. Nh of segment blockIdx.y
__global__ void __launch_bounds__(256) r2c_post_kernel(const float2* __restrict__ Z_all, const float* __restrict__ inv_asd,
                                                       float2* __restrict__ out_all, const float2* __restrict__ twF,
                                                       long long Nh) {
    const long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (j > Nh) return;
    const float2* Z = Z_all + (size_t)blockIdx.y * Nh;
    const float2 zj = Z[j == Nh ? 0 : j];
    const float2 zr = Z[j == 0 || j == Nh ? 0 : Nh - j];
    const float2 E = make_float2(0.5f * (zj.x + zr.x), 0.5f * (zj.y - zr.y));           // (Z[j] + conj Z[Nh-j]) / 2
    const float2 D = make_float2(0.5f * (zj.x - zr.x), 0.5f * (zj.y + zr.y));           // (Z[j] - conj Z[Nh-j]) / 2
    const float2 O = make_float2(D.y, -D.x);                                             // -i D
    const float2 w = j == Nh ? make_float2(-1.f, 0.f) : __ldg(twF + j);
    const float2 t = cmulf(O, w);
    float2 d = make_float2(E.x + t.x, E.y + t.y);
    if (inv_asd != nullptr) {
        const float g = __ldg(inv_asd + j);
        d.x *= g; d.y *= g;
    }
    out_all[(size_t)blockIdx.y * (Nh + 1) + j] = d;
}

}  // namespace

cudaError_t launch_r2c_table(float2* twF, long long N, cudaStream_t st) {
    r2c_table_kernel<<<(unsigned)((N / 2 + 255) / 256), 256, 0, st>>>(twF, N);
    return cudaGetLastError();
}

cudaError_t r2c_configure() {
    cudaError_t e = cudaFuncSetAttribute(r2c_pass1_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 1024 * TL * 8);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(r2c_pass2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 1024 * TL * 8);
}

// x: nb x N float32; S, Z: scratch of nb x N/2 float2 each; out: nb x (N/2+1) complex64.
cudaError_t launch_r2c(const float* x, const float* inv_asd, float2* S, float2* Z, float2* out, const float2* twF,
                       int logN, int nb, cudaStream_t st) {
    const int h = logN - 1, logA = (h + 1) / 2, logB = h / 2;
    const int A = 1 << logA, B = 1 << logB;
    const long long Nh = 1ll << h;
    r2c_pass1_kernel<<<dim3(B / TL, nb), 256, (size_t)A * TL * 8, st>>>(reinterpret_cast<const float2*>(x), S, twF, logA,
                                                                        logB, logN);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    r2c_pass2_kernel<<<dim3(A / TL, nb), 256, (size_t)B * TL * 8, st>>>(S, Z, twF, logA, logB, logN);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    r2c_post_kernel<<<dim3((unsigned)((Nh + 1 + 255) / 256), nb), 256, 0, st>>>(Z, inv_asd, out, twF, Nh);
    return cudaGetLastError();
}

}  // namespace rbmf

// =====================================================================================================================
// rbmf_prepare_strain_static (include/rbmf.h): the front end above for callers that have no device memory to give.
//
// rbmf_prepare_strain borrows three scratch arrays from the plan's workspace: the twiddle table twF (N/2 float2), the
// pass-1 intermediate S and the packed spectrum Z (n_segments N/2 float2 each).  A caller that only conditions strain
// -- a data-acquisition or whitening stage that feeds several filter processes, a plug-in that runs inside somebody
// else's pipeline and is handed nothing but its input and output buffers, a process whose framework has already
// reserved the whole card for its own pool so that a raw cudaMalloc fails, or a low-latency loop in which a cudaMalloc
// (which synchronises the device) would stall the filter streams running beside it -- has no plan, no workspace and
// no way to get either.  For them the same three kernels run on a fixed array that is part of the library image:
// it is created when the library's module is loaded on a GPU and stays until the process exits (12 MiB per GPU).
//
// The name `static_scratch` below is a real address only inside device code.  In host code it is the host-side shadow
// of the symbol; handing that to a kernel would make the kernel write through a host address.  The device address is
// looked up once per device with cudaGetSymbolAddress (static_device_state) and that pointer is what the kernels get.
// =====================================================================================================================
namespace {

constexpr long long kStaticMax = RBMF_STATIC_MAX_SAMPLES;      // samples per call, all segments together
constexpr long long kStaticPart = kStaticMax / 2;              // float2 entries of each of the three parts
// [0, kStaticPart): twF   [kStaticPart, 2 kStaticPart): S   [2 kStaticPart, 3 kStaticPart): Z
static __device__ __align__(256) float2 static_scratch[3 * kStaticPart];

constexpr int kStaticMaxDevices = 64;
struct StaticDeviceState {
    bool ready = false;
    float2* base = nullptr;   // device address of static_scratch on this device
};
std::mutex static_mutex;
StaticDeviceState static_state[kStaticMaxDevices];

// Once per device, with that device current: resolve the array's device address and raise the two passes' dynamic
// shared-memory limit (a per-device function attribute).  Neither call allocates.
cudaError_t static_device_state(float2** base) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(static_mutex);
    StaticDeviceState& s = static_state[dev];
    if (!s.ready) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, static_scratch);
        if (e != cudaSuccess) return e;
        if (p == nullptr || ((uintptr_t)p % 256) != 0) return cudaErrorInvalidSymbol;
        e = rbmf::r2c_configure();
        if (e != cudaSuccess) return e;
        s.base = static_cast<float2*>(p);
        s.ready = true;
    }
    *base = s.base;
    return cudaSuccess;
}

}  // namespace

extern "C" rbmf_status rbmf_prepare_strain_static_limits(int64_t* max_samples, size_t* scratch_bytes) {
    if (max_samples) *max_samples = kStaticMax;
    if (scratch_bytes) *scratch_bytes = sizeof(float2) * 3 * (size_t)kStaticPart;
    return RBMF_OK;
}

extern "C" rbmf_status rbmf_prepare_strain_static(const float* x_dev, const float* inv_asd_dev, int64_t N,
                                                  int32_t n_segments, void* strain_out_dev, void* cuda_stream,
                                                  int32_t* cuda_error) {
    if (cuda_error) *cuda_error = 0;
    if (!x_dev || !strain_out_dev || n_segments < 1) return RBMF_ERR_ARG;
    if (N < (1ll << 10) || N > (1ll << 24) || (N & (N - 1)) != 0) return RBMF_ERR_ARG;
    if (((uintptr_t)x_dev % 8) != 0 || ((uintptr_t)strain_out_dev % 8) != 0) return RBMF_ERR_ARG;
    // the limit: every segment of the call must fit the fixed array at once
    if (N > kStaticMax || (long long)n_segments > kStaticMax / N) return RBMF_ERR_UNSUPPORTED;
    int logN = 0;
    while ((1ll << logN) < N) ++logN;
    float2* base = nullptr;
    cudaError_t e = static_device_state(&base);
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    float2* twF = base;
    float2* S = base + kStaticPart;
    float2* Z = base + 2 * kStaticPart;
    // The array still holds whatever the previous call (any N, any stream) left in it.  Nothing here needs zeros: the
    // table is rewritten for this N on this stream, pass 1 writes every entry of S that pass 2 reads, and pass 2 every
    // entry of Z that the split reads.
    if (e == cudaSuccess) e = rbmf::launch_r2c_table(twF, N, st);
    if (e == cudaSuccess) e = rbmf::launch_r2c(x_dev, inv_asd_dev, S, Z, static_cast<float2*>(strain_out_dev), twF, logN,
                                               n_segments, st);
    if (e != cudaSuccess) {
        if (cuda_error) *cuda_error = (int32_t)e;
        return RBMF_ERR_CUDA;
    }
    return RBMF_OK;
}
