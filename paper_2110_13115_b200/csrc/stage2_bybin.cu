// Kernel 3 (step a6), by-bin version: every first-stage candidate is re-scored at full time resolution and fp32
// accuracy, with the candidates regrouped by time bin first.
//
// Why by bin.  A candidate (t, i) needs the w rows beta[i w .. i w + w) (w k complex values, 16 KB at w = 8, k = 256)
// and the coefficient row cs[t] (k values).  A loud injection lights up thousands of templates in the same few bins
// ("these triggers are not contiguous in memory"); with one warp per candidate every one of them pulls
// the same 16 KB beta block through L2 again (5 TB of L2 reads at the `large` config).  Here the list kernel 2 wrote is
// regrouped by bin with a counting sort whose histogram kernel 2's epilogue already filled:
//   stage2_alloc_kernel    one thread per bin: reserves the bin's range in the by-bin array, cuts it into work items of
//                          <= kStage2Chunk candidates, resets the counter for the scatter;
//   stage2_scatter_kernel  one thread per list entry: copies the record to its bin's range;
//   stage2_score_kernel    persistent 4-warp CTAs draw items from a ticket counter, put the item's beta block into
//                          shared memory ONCE, and each warp scores G candidates at a time against it: lane l owns the
//                          basis columns l, l + 32, ..., reads each beta value once from shared memory and uses it for
//                          all G candidates (G W complex accumulators per lane), then one halving butterfly of warp
//                          shuffles turns the 32 partial sums per output into one output per lane.
// In RBMF_GEMM_SCREEN mode the list is the fp16 screen's superset: the fp32 mean of a candidate's w samples IS the
// averaged SNR of Eq. 9 (linearity), so the stage-1 test is repeated on it at fp32 accuracy and
// the confirmed candidates go to their own list before the thr_stage2 test.
// Batches: a bin index runs over all segments, bin = b Mseg + i, and time_index = bin w + r = b N + n.
#include <mutex>

#include "rbmf_internal.h"

namespace rbmf {

namespace {

constexpr int CH = kStage2Chunk;
constexpr int NWARP = 4;
constexpr int TBUF = 128;   // staged triggers per warp (flushed above 96)
constexpr int CBUF = 64;    // staged confirmed candidates per warp (flushed above 32)

__global__ void __launch_bounds__(256) stage2_alloc_kernel(const Stage2Args a) {
    const int stride = gridDim.x * blockDim.x;
    for (int bin = blockIdx.x * blockDim.x + threadIdx.x; bin < a.Mtot; bin += stride) {
        const unsigned c = a.bin_count[bin];
        if (c == 0) continue;
        const unsigned start = (unsigned)atomicAdd(a.counters + 3, (unsigned long long)c);
        a.bin_start[bin] = start;
        a.bin_count[bin] = 0;   // the scatter counts it up again
        const unsigned nit = (c + CH - 1) / CH;
        const unsigned long long ib = atomicAdd(a.counters + 4, (unsigned long long)nit);
        for (unsigned j = 0; j < nit; ++j) {
            const unsigned left = c - j * CH;
            a.items[ib + j] = make_int4(bin, (int)(start + j * CH), (int)(left < (unsigned)CH ? left : (unsigned)CH), 0);
        }
    }
}

__global__ void __launch_bounds__(256) stage2_scatter_kernel(const Stage2Args a) {
    unsigned long long n = a.counters[0];
    if (n > a.cand_cap) n = a.cand_cap;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    const int4* src = reinterpret_cast<const int4*>(a.cand);
    int4* dst = reinterpret_cast<int4*>(a.sorted);
    for (unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const int4 cd = src[i];   // {template, bin, re, im}
        const unsigned pos = a.bin_start[cd.y] + atomicAdd(a.bin_count + cd.y, 1u);
        dst[pos] = cd;
    }
}

// Sum v[] over the 32 lanes by halving: after the five steps lane l holds the totals of entries l NV/32 .. in v[0 ..).
template <int NV>
__device__ __forceinline__ void lane_reduce(float (&v)[NV], int lane) {
#pragma unroll
    for (int s = 0; s < 5; ++s) {
        const int b = 16 >> s, h = NV >> (s + 1);
        const bool up = (lane & b) != 0;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            const float send = up ? v[i] : v[i + h];
            const float keep = up ? v[i + h] : v[i];
            v[i] = keep + __shfl_xor_sync(0xffffffffu, send, b);
        }
    }
}

// CU = basis-column steps (of 32 columns) whose coefficient loads are issued together: the G CU loads per lane come
// from L2 (~700 cycles) and must be in flight while the previous step's 4 G W FMAs run.
template <int W, int G, int CU>
__global__ void __launch_bounds__(NWARP * 32, 4) stage2_score_kernel(const Stage2Args a) {
    constexpr int NV = G * W * 2;
    static_assert(NV == 32 || NV == 64, "G W must be 16 or 32");
    extern __shared__ float4 smem4[];
    float2* sB = reinterpret_cast<float2*>(smem4);   // [W][KPP]: the item's beta block
    __shared__ rbmf_trigger tbuf_all[NWARP][TBUF];
    __shared__ rbmf_candidate cbuf_all[NWARP][CBUF];
    __shared__ unsigned long long s_item;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    rbmf_trigger* tbuf = tbuf_all[warp];
    rbmf_candidate* cbuf = cbuf_all[warp];
    int tcount = 0, ccount = 0;   // warp-uniform fill levels
    auto flush_triggers = [&]() {
        unsigned long long base = 0;
        if (lane == 0) {
            base = atomicAdd(a.trig_counter, (unsigned long long)tcount);
            if (a.trig_counter != a.counters + 1) atomicAdd(a.counters + 1, (unsigned long long)tcount);
        }
        base = __shfl_sync(0xffffffffu, base, 0);
        __syncwarp();
        for (int i = lane; i < tcount; i += 32)
            if (base + i < a.trig_cap) a.out[base + i] = tbuf[i];
        __syncwarp();
        tcount = 0;
    };
    auto flush_confirmed = [&]() {
        unsigned long long base = 0;
        if (lane == 0) base = atomicAdd(a.counters + 2, (unsigned long long)ccount);
        base = __shfl_sync(0xffffffffu, base, 0);
        __syncwarp();
        for (int i = lane; i < ccount; i += 32)
            if (base + i < a.cand_cap) a.confirmed[base + i] = cbuf[i];
        __syncwarp();
        ccount = 0;
    };

    const int k = a.k, KP = (k + 31) & ~31, KPP = KP + 2;   // row stride: + 2 keeps the float4 stores of the fill spread over banks
    const unsigned long long n_items = a.counters[4];
    const size_t chunk_stride = (size_t)a.N * kFftC;   // float2 entries between chunks of 4 columns
    const float inv_w = 1.0f / (float)W;

    for (;;) {
        __syncthreads();   // every warp is done with sB and s_item of the previous item
        if (threadIdx.x == 0) s_item = atomicAdd(a.counters + 5, 1ull);
        __syncthreads();
        const unsigned long long it = s_item;
        if (it >= n_items) break;
        const int4 item = a.items[it];
        const int bin = item.x, seg = bin / a.Mseg, ibin = bin - seg * a.Mseg;
        // ---- the bin's beta block -> shared memory: per chunk of 4 columns, W rows x 32 bytes are contiguous
        {
            const float2* brow = a.beta + (size_t)seg * a.seg_stride + (size_t)ibin * W * kFftC;
            const int total4 = (k / kFftC) * W * 2;
            for (int e = threadIdx.x; e < total4; e += NWARP * 32) {
                const int ch = e / (2 * W), rem = e - ch * (2 * W), r = rem >> 1, h = rem & 1;
                const float4 v = __ldg(reinterpret_cast<const float4*>(brow + ch * chunk_stride + r * kFftC + 2 * h));
                *reinterpret_cast<float4*>(sB + r * KPP + ch * kFftC + 2 * h) = v;
            }
            if (KP != k)
                for (int e = threadIdx.x; e < W * (KP - k); e += NWARP * 32)
                    sB[(e / (KP - k)) * KPP + k + e % (KP - k)] = make_float2(0.f, 0.f);
        }
        __syncthreads();

        const int ngroups = (item.z + G - 1) / G;
        for (int grp = warp; grp < ngroups; grp += NWARP) {
            const int nvalid = min(G, item.z - grp * G);
            const int myc = lane % G;
            const int my_t = reinterpret_cast<const int4*>(a.sorted)[item.y + grp * G + (myc < nvalid ? myc : 0)].x;
            int tg[G];
#pragma unroll
            for (int g = 0; g < G; ++g) tg[g] = __shfl_sync(0xffffffffu, my_t, g);
            float v[NV];
#pragma unroll
            for (int i = 0; i < NV; ++i) v[i] = 0.f;
#pragma unroll 1
            for (int c0 = 0; c0 < KP / 32; c0 += CU) {
                float2 cv[CU][G];
#pragma unroll
                for (int u = 0; u < CU; ++u) {
                    const int kk = lane + 32 * (c0 + u);
#pragma unroll
                    for (int g = 0; g < G; ++g)
                        cv[u][g] = kk < k ? __ldg(a.cs + (size_t)tg[g] * k + kk) : make_float2(0.f, 0.f);
                }
#pragma unroll
                for (int u = 0; u < CU; ++u) {
                    const int kk = lane + 32 * (c0 + u);
                    float2 bv[W];
#pragma unroll
                    for (int r = 0; r < W; ++r) bv[r] = sB[r * KPP + kk];
#pragma unroll
                    for (int g = 0; g < G; ++g) {
#pragma unroll
                        for (int r = 0; r < W; ++r) {
                            float& re = v[(g * W + r) * 2];
                            float& im = v[(g * W + r) * 2 + 1];
                            re = fmaf(cv[u][g].x, bv[r].x, re); re = fmaf(-cv[u][g].y, bv[r].y, re);
                            im = fmaf(cv[u][g].x, bv[r].y, im); im = fmaf(cv[u][g].y, bv[r].x, im);
                        }
                    }
                }
            }
            lane_reduce<NV>(v, lane);
            // lane -> output pair p = (g, r): NV = 64: p = lane, (re, im) = v[0], v[1];
            //                               NV = 32: entry `lane` = pair lane / 2, component lane & 1
            float re, im;
            int p;
            bool owner;
            if (NV == 64) {
                re = v[0]; im = v[1]; p = lane; owner = true;
            } else {
                const float other = __shfl_xor_sync(0xffffffffu, v[0], 1);
                re = (lane & 1) ? other : v[0]; im = (lane & 1) ? v[0] : other; p = lane >> 1; owner = (lane & 1) == 0;
            }
            const int g = p / W, r = p % W;
            const int t = __shfl_sync(0xffffffffu, my_t, g);
            bool pass = g < nvalid;
            if (a.screen) {
                // the mean of the candidate's W samples = its averaged SNR (Eq. 9): repeat the stage-1 test in fp32
                constexpr int step = NV == 64 ? 1 : 2;
                float sr = re, si = im;
#pragma unroll
                for (int o = step; o < W * step; o <<= 1) {
                    sr += __shfl_xor_sync(0xffffffffu, sr, o);
                    si += __shfl_xor_sync(0xffffffffu, si, o);
                }
                sr *= inv_w; si *= inv_w;
                pass = pass && (sr * sr + si * si >= a.thr1_sq);
                const bool emit = pass && owner && r == 0;
                const unsigned bal = __ballot_sync(0xffffffffu, emit);
                if (bal) {
                    if (emit) {
                        rbmf_candidate c2;
                        c2.template_id = t; c2.bin_index = bin; c2.avg_re = sr; c2.avg_im = si;
                        cbuf[ccount + __popc(bal & ((1u << lane) - 1u))] = c2;
                    }
                    ccount += __popc(bal);
                    if (ccount > 32) flush_confirmed();
                }
            }
            const bool hit = pass && owner && (re * re + im * im >= a.thr2_sq);
            const unsigned bal = __ballot_sync(0xffffffffu, hit);
            if (bal) {
                if (hit) {
                    rbmf_trigger tr;
                    tr.template_id = t + a.template_offset; tr.time_index = bin * W + r; tr.snr_re = re; tr.snr_im = im;
                    tbuf[tcount + __popc(bal & ((1u << lane) - 1u))] = tr;
                }
                tcount += __popc(bal);
                if (tcount > TBUF - 32) flush_triggers();
            }
        }
    }
    if (tcount > 0) flush_triggers();
    if (ccount > 0) flush_confirmed();
}

template <int W, int G, int CU>
cudaError_t launch_score_cu(const Stage2Args& a, int num_sms, cudaStream_t st) {
    // Largest dynamic shared memory size this instantiation has been set up for, PER DEVICE (a function attribute
    // belongs to the device that was current when it was set: one process-wide flag left a second GPU unconfigured),
    // under a mutex so that two host threads cannot leave the record above the attribute actually in force.
    constexpr int kDevices = 64;
    static std::mutex mu;
    static int configured[kDevices] = {};
    const int want = a.smem_bytes > 48 * 1024 ? a.smem_bytes : 48 * 1024;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    {
        std::lock_guard<std::mutex> lock(mu);
        const bool known = dev >= 0 && dev < kDevices;
        if (!known || want > configured[dev]) {
            e = cudaFuncSetAttribute(stage2_score_kernel<W, G, CU>, cudaFuncAttributeMaxDynamicSharedMemorySize, want);
            if (e != cudaSuccess) return e;
            if (known) configured[dev] = want;
        }
    }
    int per_sm = (200 * 1024) / (a.smem_bytes + 14 * 1024);
    per_sm = per_sm < 1 ? 1 : (per_sm > 6 ? 6 : per_sm);
    stage2_score_kernel<W, G, CU><<<num_sms * per_sm, NWARP * 32, a.smem_bytes, st>>>(a);
    return cudaGetLastError();
}

template <int W, int G>
cudaError_t launch_score(const Stage2Args& a, int num_sms, cudaStream_t st) {
    const int steps = ((a.k + 31) & ~31) / 32;
    constexpr int CUMAX = G <= 4 ? 4 : 2;   // G CU coefficient values (2 registers each) are held at once
    if (steps % CUMAX == 0) return launch_score_cu<W, G, CUMAX>(a, num_sms, st);
    if (steps % 2 == 0) return launch_score_cu<W, G, 2>(a, num_sms, st);
    return launch_score_cu<W, G, 1>(a, num_sms, st);
}

}  // namespace

// Shared memory the score kernel needs for one bin's beta block; 0 if this (w, k) does not fit (then the
// warp-per-candidate kernel of stage2_kernels.cu is used).
int stage2_bybin_smem(int w, int k) {
    const int KPP = ((k + 31) & ~31) + 2;
    const long long bytes = (long long)w * KPP * 8;
    return bytes <= 160 * 1024 ? (int)bytes : 0;
}

cudaError_t launch_stage2_bybin(const Stage2Args& a, int num_sms, cudaStream_t st) {
    stage2_alloc_kernel<<<(a.Mtot + 255) / 256 < num_sms * 8 ? (a.Mtot + 255) / 256 : num_sms * 8, 256, 0, st>>>(a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    stage2_scatter_kernel<<<num_sms * 8, 256, 0, st>>>(a);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    switch (a.w) {
        case 1: return launch_score<1, 16>(a, num_sms, st);
        case 2: return launch_score<2, 8>(a, num_sms, st);
        case 4: return launch_score<4, 8>(a, num_sms, st);
        case 8: return launch_score<8, 4>(a, num_sms, st);
        case 16: return launch_score<16, 2>(a, num_sms, st);
        case 32: return launch_score<32, 1>(a, num_sms, st);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace rbmf
