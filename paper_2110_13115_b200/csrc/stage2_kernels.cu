// Kernel 3 (step a6): re-score every first-stage candidate at full time resolution and fp32 accuracy
// with one warp per candidate -- the fallback of the by-bin kernel (stage2_bybin.cu)
// for the (w, k) whose beta block does not fit in shared memory (w = 32 with k > 608), also selectable for tests with
// RBMF_DIAG_STAGE2_PER_CANDIDATE --, plus the plain fp32 verification version of kernel 2 (RBMF_DIAG_STAGE1_FP32_CHECK).
#include <cuda_bf16.h>

#include "rbmf_internal.h"

namespace rbmf {

// One warp per candidate (t, i): rho_t[i w + r] = sum_c cs[t][c] * beta[i w + r][c], r < w  (cs = conj(c)/sigma).
// beta is chunk-blocked, [chunk][n][C = 4]: per chunk the candidate's w rows are one contiguous block of w * 32
// bytes.  The warp walks float4 items e = (chunk, r, half) in this order, e = lane, lane + 32, ...: with 2w <= 32 a
// lane always sees the same (r, half), so it accumulates one row's partial sum; w = 32 alternates between two rows.
// Outputs are staged per warp in shared memory and flushed with ONE atomicAdd per 32+ records: with millions of
// candidates (a loud injection in a dense bank) per-candidate atomics on the two list counters serialise in L2.
__global__ void __launch_bounds__(256) stage2_kernel(const Stage2Args a) {
    __shared__ rbmf_trigger tbuf_all[8][64];
    __shared__ rbmf_candidate cbuf_all[8][32];
    rbmf_trigger* tbuf = tbuf_all[threadIdx.x >> 5];
    rbmf_candidate* cbuf = cbuf_all[threadIdx.x >> 5];
    int tcount = 0, ccount = 0;   // warp-uniform fill levels
    auto flush_triggers = [&](int lane_) {
        unsigned long long base = 0;
        if (lane_ == 0) {
            base = atomicAdd(a.trig_counter, (unsigned long long)tcount);
            if (a.trig_counter != a.counters + 1) atomicAdd(a.counters + 1, (unsigned long long)tcount);
        }
        base = __shfl_sync(0xffffffffu, base, 0);
        __syncwarp();
        for (int i = lane_; i < tcount; i += 32)
            if (base + i < a.trig_cap) a.out[base + i] = tbuf[i];
        __syncwarp();
        tcount = 0;
    };
    auto flush_confirmed = [&](int lane_) {
        unsigned long long base = 0;
        if (lane_ == 0) base = atomicAdd(a.counters + 2, (unsigned long long)ccount);
        base = __shfl_sync(0xffffffffu, base, 0);
        __syncwarp();
        if (lane_ < ccount && base + lane_ < a.cand_cap) a.confirmed[base + lane_] = cbuf[lane_];
        __syncwarp();
        ccount = 0;
    };
    const int lane = threadIdx.x & 31;
    const unsigned long long warp0 = (unsigned long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const unsigned long long nwarps = (unsigned long long)gridDim.x * (blockDim.x >> 5);
    unsigned long long n_cand = a.counters[0];
    if (n_cand > a.cand_cap) n_cand = a.cand_cap;
    const int k = a.k, w = a.w;
    const int per_chunk = 2 * w;                       // float4 items per chunk
    const int total = (k / kFftC) * per_chunk;
    const size_t chunk_stride = (size_t)a.N * kFftC;    // float2 entries
    for (unsigned long long ci = warp0; ci < n_cand; ci += nwarps) {
        const rbmf_candidate cd = a.cand[ci];
        const float2* __restrict__ crow = a.cs + (size_t)cd.template_id * k;
        const int seg = cd.bin_index / a.Mseg;   // batches: bin = segment * Mseg + i, beta arrays seg_stride apart
        const float2* __restrict__ brow = a.beta + (size_t)seg * a.seg_stride + (size_t)(cd.bin_index - seg * a.Mseg) * w * kFftC;
        float re0 = 0.f, im0 = 0.f, re1 = 0.f, im1 = 0.f;
        // per_chunk = 2w is a power of two: shifts instead of divisions; four items per lane in flight (the loop is
        // bound by the latency of its two loads, not by their bandwidth)
        const int lg = 31 - __clz(per_chunk);
        auto item = [&](int e, float& ar, float& ai) {
            const int ch = e >> lg, rem = e & (per_chunk - 1);
            const int r = rem >> 1, h = rem & 1;
            const float4 p = __ldg(reinterpret_cast<const float4*>(crow + ch * kFftC + 2 * h));
            const float4 x = __ldg(reinterpret_cast<const float4*>(brow + ch * chunk_stride + r * kFftC + 2 * h));
            float vr = p.x * x.x, vi = p.x * x.y;
            vr = fmaf(-p.y, x.y, vr); vr = fmaf(p.z, x.z, vr); vr = fmaf(-p.w, x.w, vr);
            vi = fmaf(p.y, x.x, vi); vi = fmaf(p.z, x.w, vi); vi = fmaf(p.w, x.z, vi);
            ar += vr; ai += vi;
        };
        int e = lane;
        if (per_chunk > 32) {   // w = 32: consecutive items of a lane alternate between rows r and r + 16
            for (; e + 96 < total; e += 128) {
                item(e, re0, im0); item(e + 32, re1, im1); item(e + 64, re0, im0); item(e + 96, re1, im1);
            }
            for (int par = 0; e < total; e += 32, par ^= 1) { if (par) item(e, re1, im1); else item(e, re0, im0); }
        } else {
            // a lane keeps its (row r, half h) and walks the chunks ch0, ch0 + dch, ...: two pointers, constant strides
            const int rem = lane & (per_chunk - 1), dch = 32 >> lg, nch = k / kFftC;
            const float4* pc = reinterpret_cast<const float4*>(crow + (lane >> lg) * kFftC + 2 * (rem & 1));
            const float4* px = reinterpret_cast<const float4*>(brow + (size_t)(lane >> lg) * chunk_stride +
                                                               (rem >> 1) * kFftC + 2 * (rem & 1));
            const size_t sc = (size_t)dch * kFftC / 2, sx = (size_t)dch * chunk_stride / 2;   // float4 strides
            auto mac = [&](const float4 p, const float4 x, float& ar, float& ai) {
                ar = fmaf(p.x, x.x, ar); ar = fmaf(-p.y, x.y, ar); ar = fmaf(p.z, x.z, ar); ar = fmaf(-p.w, x.w, ar);
                ai = fmaf(p.x, x.y, ai); ai = fmaf(p.y, x.x, ai); ai = fmaf(p.z, x.w, ai); ai = fmaf(p.w, x.z, ai);
            };
            float r2 = 0.f, i2 = 0.f, r3 = 0.f, i3 = 0.f;
            int ch = lane >> lg;
            for (; ch + 3 * dch < nch; ch += 4 * dch, pc += 4 * sc, px += 4 * sx) {
                const float4 p0 = __ldg(pc), p1 = __ldg(pc + sc), p2 = __ldg(pc + 2 * sc), p3 = __ldg(pc + 3 * sc);
                const float4 x0 = __ldg(px), x1 = __ldg(px + sx), x2 = __ldg(px + 2 * sx), x3 = __ldg(px + 3 * sx);
                mac(p0, x0, re0, im0); mac(p1, x1, re1, im1); mac(p2, x2, r2, i2); mac(p3, x3, r3, i3);
            }
            for (; ch < nch; ch += dch, pc += sc, px += sx) mac(__ldg(pc), __ldg(px), re0, im0);
            re0 += re1 + r2 + r3; im0 += im1 + i2 + i3;
            re1 = 0.f; im1 = 0.f;
        }
        // lanes that share a row differ in bit 0 (half) and in the bits >= log2(2w)
        for (int o = 1; o < 32; o <<= 1) {
            if (o == 1 || o >= per_chunk) {
                re0 += __shfl_xor_sync(0xffffffffu, re0, o); im0 += __shfl_xor_sync(0xffffffffu, im0, o);
                re1 += __shfl_xor_sync(0xffffffffu, re1, o); im1 += __shfl_xor_sync(0xffffffffu, im1, o);
            }
        }
        // even lane 2r < 2w holds row r (and row 16 + r in slot 1 when w = 32)
        const int nslot = per_chunk > 32 ? 2 : 1;
        if (a.screen) {
            // `cand` is the fp16 screen's superset: the fp32 average of the w samples IS the averaged SNR of Eq. 9
            // (linearity), so the stage-1 test is repeated here at fp32 accuracy.
            const bool own = (lane & 1) == 0 && lane < per_chunk;
            float sr = own ? re0 + (nslot == 2 ? re1 : 0.f) : 0.f;
            float si = own ? im0 + (nslot == 2 ? im1 : 0.f) : 0.f;
            for (int o = 16; o > 0; o >>= 1) {
                sr += __shfl_xor_sync(0xffffffffu, sr, o);
                si += __shfl_xor_sync(0xffffffffu, si, o);
            }
            const float inv_w = 1.0f / (float)w;
            sr *= inv_w; si *= inv_w;
            if (!(sr * sr + si * si >= a.thr1_sq)) continue;   // warp-uniform
            if (lane == 0) {
                rbmf_candidate c2;
                c2.template_id = cd.template_id; c2.bin_index = cd.bin_index; c2.avg_re = sr; c2.avg_im = si;
                cbuf[ccount] = c2;
            }
            if (++ccount == 32) flush_confirmed(lane);
        }
        for (int s = 0; s < nslot; ++s) {
            const int r = (lane >> 1) + 16 * s;
            const float vr = s ? re1 : re0, vi = s ? im1 : im0;
            const bool owner = (lane & 1) == 0 && lane < per_chunk;
            const bool hit = owner && (vr * vr + vi * vi >= a.thr2_sq);
            const unsigned ballot = __ballot_sync(0xffffffffu, hit);
            if (ballot) {
                if (hit) {
                    rbmf_trigger t;
                    t.template_id = cd.template_id + a.template_offset;
                    t.time_index = cd.bin_index * w + r;
                    t.snr_re = vr;
                    t.snr_im = vi;
                    tbuf[tcount + __popc(ballot & ((1u << lane) - 1u))] = t;
                }
                tcount += __popc(ballot);          // at most 16 per slot: 32 + 16 <= 64 entries
                if (tcount > 32) flush_triggers(lane);
            }
        }
    }
    if (tcount > 0) flush_triggers(lane);
    if (ccount > 0) flush_confirmed(lane);
}

cudaError_t launch_stage2(const Stage2Args& a, int num_sms, cudaStream_t st) {
    stage2_kernel<<<num_sms * 8, 256, 0, st>>>(a);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Verification version of steps a4-a5 on CUDA cores: the same bf16 hi/lo operand planes as the tensor-core
// kernel, recombined to fp32 (hi + lo) and multiplied in fp32.  64 time bins x 64 templates per CTA.
__device__ __forceinline__ float plane_val(const uint16_t* hi, const uint16_t* lo, size_t e) {
    return __bfloat162float(__ushort_as_bfloat16(hi[e])) + __bfloat162float(__ushort_as_bfloat16(lo[e]));
}

__global__ void __launch_bounds__(256) gemm_simt_kernel(const uint16_t* __restrict__ a_hi,
                                                        const uint16_t* __restrict__ a_lo,
                                                        const uint16_t* __restrict__ c_hi,
                                                        const uint16_t* __restrict__ c_lo, const GemmArgs g,
                                                        const int Mplane) {
    constexpr int TI = 64, TT = 64, KB = 32;
    __shared__ float sA[TI][KB + 1];       // beta^avg rows (time bins) x K
    __shared__ float sRe[TT][KB + 1];      // template "re" rows
    __shared__ float sIm[TT][KB + 1];      // template "im" rows
    const int i0 = blockIdx.y * TI, t0 = blockIdx.x * TT;   // templates on grid.x (up to 2^24 of them)
    const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;   // 16 x 16 threads, 4 x 4 outputs each
    float re[4][4] = {}, im[4][4] = {};
    for (int k0 = 0; k0 < g.k2; k0 += KB) {
        for (int e = threadIdx.x; e < TI * KB; e += 256) {
            const int r = e / KB, kk = e % KB;
            const int i = i0 + r;
            sA[r][kk] = i < g.M ? plane_val(a_hi, a_lo, ((size_t)((k0 + kk) / 64) * Mplane + i) * 64 + (k0 + kk) % 64) : 0.f;
            const int t = t0 + r;   // t < Tpad always (grid covers padded templates)
            const size_t row_re = (size_t)(t / kGemmTT) * 2 * kGemmTT + (t % kGemmTT);
            sRe[r][kk] = plane_val(c_hi, c_lo, row_re * g.k2 + k0 + kk);
            sIm[r][kk] = plane_val(c_hi, c_lo, (row_re + kGemmTT) * g.k2 + k0 + kk);
        }
        __syncthreads();
#pragma unroll 4
        for (int kk = 0; kk < KB; ++kk) {
            float av[4], rv[4], iv[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { av[u] = sA[ty * 4 + u][kk]; rv[u] = sRe[tx * 4 + u][kk]; iv[u] = sIm[tx * 4 + u][kk]; }
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int v = 0; v < 4; ++v) { re[u][v] = fmaf(av[u], rv[v], re[u][v]); im[u][v] = fmaf(av[u], iv[v], im[u][v]); }
        }
        __syncthreads();
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int v = 0; v < 4; ++v) {
            const int i = i0 + ty * 4 + u, t = t0 + tx * 4 + v;
            if (i < g.M && t < g.T && re[u][v] * re[u][v] + im[u][v] * im[u][v] >= g.thr1_sq) {
                const unsigned long long idx = atomicAdd(g.counters, 1ULL);
                if (idx < g.cand_cap) {
                    rbmf_candidate cd;
                    cd.template_id = t; cd.bin_index = i; cd.avg_re = re[u][v]; cd.avg_im = im[u][v];
                    g.cand[idx] = cd;
                    atomicAdd(g.bin_count + i, 1u);
                }
            }
        }
}

cudaError_t launch_gemm_simt(const uint16_t* a_hi, const uint16_t* a_lo, const uint16_t* c_hi, const uint16_t* c_lo,
                             const GemmArgs& g, int Mplane, cudaStream_t st) {
    dim3 grid((unsigned)(g.num_tb * kGemmTT / 64), (unsigned)((g.M + 63) / 64));
    gemm_simt_kernel<<<grid, 256, 0, st>>>(a_hi, a_lo, c_hi, c_lo, g, Mplane);
    return cudaGetLastError();
}

}  // namespace rbmf
