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

template <int D>
__global__ void __launch_bounds__(kAttnWarps * 32) llx_attn_partial(const AttnArgs a) {
    constexpr int LPH = D / 8;    // lanes per head
    constexpr int HPW = 32 / LPH; // heads per warp
    const int b = blockIdx.z;
    const int split = blockIdx.x;
    const int ctx = a.ctx_lens[b];
    const int t0 = split * a.split_tokens;
    if (t0 >= ctx) return;
    const int t1 = min(ctx, t0 + a.split_tokens);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int h = (blockIdx.y * kAttnWarps + warp) * HPW + lane / LPH;
    const int dl = (lane % LPH) * 8;  // first dim owned by this lane
    const bool head_ok = h < a.H;
    const int hc = head_ok ? h : a.H - 1;  // clamp: idle lanes still take part in the shuffles

    float qf[8];
    unpack8(*reinterpret_cast<const uint4*>(a.q + ((long long)b * a.H + hc) * D + dl), qf);
#pragma unroll
    for (int j = 0; j < 8; ++j) qf[j] *= a.scale_log2;

    const long long row_bytes = (long long)a.H * D * 2;  // one token, all heads
    const long long lane_off = ((long long)hc * D + dl) * 2;
    const int32_t* bt = a.block_tables + (long long)b * a.max_blocks;

    float m = -INFINITY, l = 0.f, acc[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[j] = 0.f;

    for (int t = t0; t < t1; t += kAttnGroup) {
        uint4 kq[kAttnGroup], vq[kAttnGroup];
#pragma unroll
        for (int g = 0; g < kAttnGroup; ++g) {
            const int tt = t + g;
            if (tt < t1) {
                const int blk = __ldg(bt + tt / a.S);
                const long long off = blk * a.tile_bytes + (long long)(tt % a.S) * row_bytes + lane_off;
                kq[g] = ld_kv16(a.k_base + off);
                vq[g] = ld_kv16(a.v_base + off);
            } else {
                kq[g] = make_uint4(0, 0, 0, 0);
                vq[g] = make_uint4(0, 0, 0, 0);
            }
        }
        float s[kAttnGroup];
        float gmax = -INFINITY;
#pragma unroll
        for (int g = 0; g < kAttnGroup; ++g) {
            float kf[8];
            unpack8(kq[g], kf);
            float d = 0.f;
#pragma unroll
            for (int j = 0; j < 8; ++j) d = fmaf(qf[j], kf[j], d);
#pragma unroll
            for (int o = LPH / 2; o >= 1; o >>= 1) d += __shfl_xor_sync(0xffffffffu, d, o);
            s[g] = (t + g < t1) ? d : -INFINITY;
            gmax = fmaxf(gmax, s[g]);
        }
        const float m_new = fmaxf(m, gmax);  // finite: the group holds at least one valid token
        const float corr = exp2f(m - m_new);
        l *= corr;
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[j] *= corr;
#pragma unroll
        for (int g = 0; g < kAttnGroup; ++g) {
            const float p = exp2f(s[g] - m_new);
            float vf[8];
            unpack8(vq[g], vf);
            l += p;
#pragma unroll
            for (int j = 0; j < 8; ++j) acc[j] = fmaf(p, vf[j], acc[j]);
        }
        m = m_new;
    }
    if (!head_ok) return;
    float* o = a.part + (((long long)b * a.H + h) * a.max_splits + split) * (D + 4);
    *reinterpret_cast<float4*>(o + dl) = make_float4(acc[0], acc[1], acc[2], acc[3]);
    *reinterpret_cast<float4*>(o + dl + 4) = make_float4(acc[4], acc[5], acc[6], acc[7]);
    if ((lane % LPH) == 0) {
        o[D] = m;
        o[D + 1] = l;
    }
}

// grid (H, B), D threads: out[b][h][d] = sum_s 2^(m_s-M) acc_s[d] / sum_s 2^(m_s-M) l_s
template <int D>
__global__ void __launch_bounds__(D) llx_attn_merge(const AttnArgs a) {
    const int h = blockIdx.x, b = blockIdx.y, d = threadIdx.x;
    const int ctx = a.ctx_lens[b];
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
