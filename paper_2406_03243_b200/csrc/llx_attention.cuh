// Stand-in paged decode attention (S7): one query token per sequence, MHA, fp16 in,
// fp32 accumulate, fp16 out.  The standard KV-cache attention the paper builds on
// (§2) read through a block table (PagedAttention).  It exists
// to measure how much a concurrent migration slows a decode step (§6.2).
//
//   o[b][h] = sum_t softmax_t(scale * q[b][h].k_t[h]) v_t[h],   t < ctx_len[b]
//
// HBM-bound (K and V are read once, ~0.5 flop/byte), so the design is about contiguous reads:
// in the pool layout [block][slot][head][dim] the heads of one token are adjacent, so a CTA of
// 8 warps covers 8*HPW adjacent heads (HPW = heads per warp = 256/head_dim... see below) and
// reads 8*HPW*head_dim*2 contiguous bytes of K (and of V) per token.  Work is split along the
// context (flash-decoding): CTA (split, head group, sequence) reduces `split_tokens` tokens
// with an online softmax and writes an unnormalised partial (m, l, acc[D]) in fp32; a second
// kernel merges the partials with the log-sum-exp rescale and rounds to fp16 (RNE).
//
// Lane mapping: each lane owns 8 consecutive dims (one 16-byte load); LPH = D/8 lanes form a
// head, a warp holds HPW = 32/LPH heads.  Scores are reduced over the LPH lanes by xor-shuffles.
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace llx {

struct AttnArgs {
    const unsigned char* k_base;  // pool[layer][0][0]
    const unsigned char* v_base;  // pool[layer][1][0]
    const __half* q;              // [B,H,D]
    __half* out;                  // [B,H,D]
    const int32_t* block_tables;  // [B,max_blocks]
    const int32_t* ctx_lens;      // [B]
    float* part;                  // [B][H][max_splits][D+4] : acc[D], m, l, pad (16-byte rows)
    long long tile_bytes;
    int H, S, max_blocks, max_splits, split_tokens;
    float scale_log2;  // scale * log2(e): softmax is evaluated with exp2
};

constexpr int kAttnWarps = 8;
constexpr int kAttnGroup = 8;  // tokens whose K and V loads are in flight together per lane

__device__ __forceinline__ uint4 ld_kv16(const void* p) {
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void unpack8(const uint4& u, float* f) {
    const __half2* h = reinterpret_cast<const __half2*>(&u);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        float2 t = __half22float2(h[j]);
        f[2 * j] = t.x;
        f[2 * j + 1] = t.y;
    }
}

// two fp32 FMAs per instruction (sm_100 FFMA2): c += a * b on float2
__device__ __forceinline__ void ffma2(float2& c, const float2 a, const float2 b) {
    unsigned long long ra, rb, rc;
    asm("mov.b64 %0, {%1,%2};" : "=l"(ra) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1,%2};" : "=l"(rb) : "f"(b.x), "f"(b.y));
    asm("mov.b64 %0, {%1,%2};" : "=l"(rc) : "f"(c.x), "f"(c.y));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(rc) : "l"(ra), "l"(rb));
    asm("mov.b64 {%0,%1}, %2;" : "=f"(c.x), "=f"(c.y) : "l"(rc));
}

__device__ __forceinline__ void griddep_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void griddep_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <int D>
__global__ void __maxnreg__(112) llx_attn_partial(const AttnArgs a) {
    constexpr int LPH = D / 8;     // lanes per head
    constexpr int HPW = 32 / LPH;  // heads per warp
    constexpr int G = kAttnGroup;  // 8 tokens per group
    static_assert(G == 8 && LPH >= 8, "the transposed reduction below assumes 8 tokens and >= 8 lanes per head");
    griddep_wait();
    const int b = blockIdx.z;
    const int split = blockIdx.x;
    const int ctx = min(a.ctx_lens[b], a.max_blocks * a.S);  // llx.h: a longer ctx_len is clamped, never followed past the table row
    const int t0 = split * a.split_tokens;
    if (t0 >= ctx) return;
    const int t1 = min(ctx, t0 + a.split_tokens);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int li = lane % LPH;  // lane within its head
    const int h = (blockIdx.y * kAttnWarps + warp) * HPW + lane / LPH;
    const int dl = li * 8;  // first dim owned by this lane
    const bool head_ok = h < a.H;
    const int hc = head_ok ? h : a.H - 1;  // clamp: idle lanes still take part in the shuffles

    float2 q2[4];
    {
        const uint4 qu = *reinterpret_cast<const uint4*>(a.q + ((long long)b * a.H + hc) * D + dl);
        const __half2* qh = reinterpret_cast<const __half2*>(&qu);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            q2[j] = __half22float2(qh[j]);
            q2[j].x *= a.scale_log2;
            q2[j].y *= a.scale_log2;
        }
    }
    const long long row_bytes = (long long)a.H * D * 2;  // one token, all heads
    const long long lane_off = ((long long)hc * D + dl) * 2;
    const int32_t* bt = a.block_tables + (long long)b * a.max_blocks;

    // halving offsets of the transposed reduction: after them this lane owns the score of token g_own
    constexpr int O1 = LPH / 2, O2 = LPH / 4, O3 = LPH / 8;
    const bool b1 = li & O1, b2 = li & O2, b3 = li & O3;
    const int g_own = (b1 ? 4 : 0) + (b2 ? 2 : 0) + (b3 ? 1 : 0);

    float m = -INFINITY, l = 0.f;  // l: partial over the tokens this lane owned
    float2 acc[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) acc[j] = make_float2(0.f, 0.f);

    int bi = t0 / a.S;
    int blk_first = bi * a.S;  // token index of slot 0 of block bi
    for (; blk_first < t1; ++bi, blk_first += a.S) {
        const int blk = __ldg(bt + bi);
        const int s_lo = max(t0 - blk_first, 0);
        const int s_hi = min(t1 - blk_first, a.S);
        const unsigned char* kb = a.k_base + blk * a.tile_bytes + lane_off;
        const unsigned char* vb = a.v_base + blk * a.tile_bytes + lane_off;
        for (int s0 = s_lo; s0 < s_hi; s0 += G) {
            const int nvalid = s_hi - s0;  // >= 1; tokens g >= nvalid are masked
            uint4 kq[G], vq[G];
#pragma unroll
            for (int g = 0; g < G; ++g) {
                if (g < nvalid) {
                    const long long off = (long long)(s0 + g) * row_bytes;
                    kq[g] = ld_kv16(kb + off);
                    vq[g] = ld_kv16(vb + off);
                } else {
                    kq[g] = make_uint4(0, 0, 0, 0);
                    vq[g] = make_uint4(0, 0, 0, 0);
                }
            }
            // partial dot products of this lane's 8 dims with each of the 8 tokens
            float d[G];
#pragma unroll
            for (int g = 0; g < G; ++g) {
                const __half2* kh = reinterpret_cast<const __half2*>(&kq[g]);
                float2 s2 = make_float2(0.f, 0.f);
#pragma unroll
                for (int j = 0; j < 4; ++j) ffma2(s2, q2[j], __half22float2(kh[j]));
                d[g] = s2.x + s2.y;
            }
            // transposed reduction over the LPH lanes: 4 + 2 + 1 shuffles instead of 8 * log2(LPH)
            float k4[4], k2[2], sc;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float mine = b1 ? d[4 + j] : d[j], other = b1 ? d[j] : d[4 + j];
                k4[j] = mine + __shfl_xor_sync(0xffffffffu, other, O1);
            }
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const float mine = b2 ? k4[2 + j] : k4[j], other = b2 ? k4[j] : k4[2 + j];
                k2[j] = mine + __shfl_xor_sync(0xffffffffu, other, O2);
            }
            {
                const float mine = b3 ? k2[1] : k2[0], other = b3 ? k2[0] : k2[1];
                sc = mine + __shfl_xor_sync(0xffffffffu, other, O3);
            }
#pragma unroll
            for (int o = O3 / 2; o >= 1; o >>= 1) sc += __shfl_xor_sync(0xffffffffu, sc, o);
            if (g_own >= nvalid) sc = -INFINITY;
            // online softmax: group max over the head's lanes, one exp2 per lane
            float gmax = sc;
            gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, O1));
            gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, O2));
            gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, O3));
            const float m_new = fmaxf(m, gmax);  // finite: token s0 is valid
            const float corr = exp2f(m - m_new);
            const float p_own = exp2f(sc - m_new);
            l = l * corr + p_own;
            m = m_new;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                acc[j].x *= corr;
                acc[j].y *= corr;
            }
#pragma unroll
            for (int g = 0; g < G; ++g) {
                // the lane (within the head) that owns token g: bits of g placed at O1, O2, O3
                const int src = ((g & 4) ? O1 : 0) + ((g & 2) ? O2 : 0) + ((g & 1) ? O3 : 0);
                const float p = __shfl_sync(0xffffffffu, p_own, src, LPH);
                const float2 p2 = make_float2(p, p);
                const __half2* vh = reinterpret_cast<const __half2*>(&vq[g]);
#pragma unroll
                for (int j = 0; j < 4; ++j) ffma2(acc[j], p2, __half22float2(vh[j]));
            }
        }
    }
    // dependents may start launching now: triggering only after the main loop keeps waiting CTAs of the next
    // kernel from occupying registers while this kernel still needs both of its CTAs per SM (measured: an early
    // trigger costs +25 % under a concurrent full-width migration)
    griddep_launch();
    // l: sum over the distinct token owners (lanes differing in the O1, O2, O3 bits)
    l += __shfl_xor_sync(0xffffffffu, l, O1);
    l += __shfl_xor_sync(0xffffffffu, l, O2);
    l += __shfl_xor_sync(0xffffffffu, l, O3);
    if (!head_ok) return;
    float* o = a.part + (((long long)b * a.H + h) * a.max_splits + split) * (D + 4);
    *reinterpret_cast<float4*>(o + dl) = make_float4(acc[0].x, acc[0].y, acc[1].x, acc[1].y);
    *reinterpret_cast<float4*>(o + dl + 4) = make_float4(acc[2].x, acc[2].y, acc[3].x, acc[3].y);
    if (li == 0) {
        o[D] = m;
        o[D + 1] = l;
    }
}

// grid (H, B), D threads: out[b][h][d] = sum_s 2^(m_s-M) acc_s[d] / sum_s 2^(m_s-M) l_s
template <int D>
__global__ void __launch_bounds__(D) llx_attn_merge(const AttnArgs a) {
    griddep_wait();    // wait first, then let dependents launch (llx_copy.cuh, ring_copy): a kernel behind this one
    griddep_launch();  // never starts before llx_attn_partial has completed
    const int h = blockIdx.x, b = blockIdx.y, d = threadIdx.x;
    const int ctx = min(a.ctx_lens[b], a.max_blocks * a.S);  // llx.h: a longer ctx_len is clamped, never followed past the table row
    const int ns = (ctx + a.split_tokens - 1) / a.split_tokens;
    const float* p = a.part + ((long long)b * a.H + h) * a.max_splits * (D + 4);
    float M = -INFINITY;
    for (int s = 0; s < ns; ++s) M = fmaxf(M, p[s * (D + 4) + D]);
    float num = 0.f, den = 0.f;
    for (int s = 0; s < ns; ++s) {
        const float w = exp2f(p[s * (D + 4) + D] - M);
        num = fmaf(w, p[s * (D + 4) + d], num);
        den = fmaf(w, p[s * (D + 4) + D + 1], den);
    }
    a.out[((long long)b * a.H + h) * D + d] = __float2half_rn(ns > 0 ? num / den : 0.f);
}

}  // namespace llx
