// sc_attn_decode.cu -- paged attention for a FEW new tokens per conversation (decode, n = 1; short
// speculative or chunk tails), SURVEY.md 8(f) row f4 "decode (n = 1) over the pool", PAPER.md:382 (TPOT);
// the operation is the same as a6: row i attends to keys 0 .. T_h + i.
//
// With one to a few query rows the path is a pure paged READ of the history: 4 D flops per key and
// head against 4 D bytes of K and V, so the bound is HBM and the kernel is built around keeping bytes in
// flight, not around the tensor pipe (the prefill kernel's 256-row CTA keeps 2-3 of its five 32 KiB slots
// busy because its producer paces itself on the MMA chain: 0.39 of HBM at 5 120 tokens):
//   * one CTA per (split of the keys, KV head, conversation); the query rows of ALL query heads of the
//     group and all new tokens of the conversation (at most 16 rows = n * Hq/Hkv) share one pass over
//     that KV head's chunks, so grouped-query models read K/V once per group;
//   * a 3-stage ring of 64-token tiles (K and V chunks of 4 pool blocks, 32 KiB at D = 128) filled with
//     cp.async 16-byte copies by all 128 threads; two CTAs per SM keep 4 tiles = 128 KiB in flight per
//     SM, above the ~64 KiB an SM needs to draw its share of HBM;
//   * the arithmetic is one m16n8k16 mma.sync row block: the 16 (padded) rows against the 16 tokens
//     of one pool block per warp -- warp w owns block w of every tile -- with the usual online softmax
//     in registers; it is a few hundred cycles per 32 KiB tile;
//   * the four warps' (m, l, O) are merged through shared memory at the end, added in a fixed order
//     (deterministic); with several splits the CTA writes the fp32 partial in the layout
//     sc_combine_kernel reads (sc_attn_mma.cu).
// The new tokens' K/V are scattered by sc_scatter_read_kernel before this kernel (sc_ops.cu).
// Work partitioning depends on logical positions only: results do not depend on physical block ids.
#include <cuda_bf16.h>

#include "sc_internal.h"

namespace {

constexpr int kRows = 16;      // query rows per CTA: (new token, query head of the group) pairs
constexpr int kTileN = 64;     // KV tokens per tile (4 pool blocks, one per warp)
constexpr int kThreads = 128;
constexpr int kStages = 3;

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma_bf16(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1)
{
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, "
        "{%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&v);
}

template <int D>
__global__ void __launch_bounds__(kThreads, 2)
sc_attn_decode_kernel(ScGeom g, ScBatch b, ScAttnArgs a)
{
    constexpr int kChunk = 16 * D * 2;            // bytes of one (block, head) chunk
    constexpr int kStage = 8 * kChunk;            // K: 4 chunks, V: 4 chunks
    constexpr int NH = D / 64;
    constexpr int KS = D / 16;                    // k-steps of QK^T
    constexpr int DB = D / 8;                     // n-blocks of O
    extern __shared__ __align__(1024) char smem[];

    const int split = blockIdx.x, hk = blockIdx.y, s = blockIdx.z;
    const int n_s = b.cu_new[s + 1] - b.cu_new[s];
    if (n_s == 0) return;
    const int G = g.Hq / g.Hkv;
    const int R = n_s * G;                        // valid rows: row r = (token r / G, query head hk*G + r % G)
    const int T_h = b.hist[s];
    const int kmax = T_h + n_s;                   // keys [0, kmax) are visible to the last row
    const int tiles_needed = (kmax + kTileN - 1) / kTileN;
    const int t_begin = split * a.split_units;
    const int t_end = min(t_begin + a.split_units, tiles_needed);
    if (t_begin >= t_end) return;
    const int nblk_s = (kmax + 15) >> 4;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int gq = lane >> 2, tq = lane & 3;

    auto load_tile = [&](int jt, int st) {
        char *dst = smem + st * kStage;
#pragma unroll
        for (int ci = 0; ci < 8; ++ci) {
            const int kvsel = ci >> 2, blk = ci & 3;
            const int lb = min(jt * 4 + blk, nblk_s - 1);      // past the end: the last block again (masked)
            const char *src = a.kv.base + sc_phys_block(a.kv, b, s, lb) * a.kv.block_stride +
                              (int64_t)(kvsel * g.Hkv + hk) * kChunk;
#pragma unroll
            for (int off = tid * 16; off < kChunk; off += kThreads * 16)
                cp_async16(smem_u32(dst + ci * kChunk + off), src + off);
        }
    };
    // the ring is filled first: kStages - 1 tiles are requested before anything else is done
#pragma unroll
    for (int st = 0; st < kStages - 1; ++st) {
        if (t_begin + st < t_end) load_tile(t_begin + st, st);
        asm volatile("cp.async.commit_group;" ::: "memory");
    }

    // ---- Q fragments straight from global (once per CTA; every warp holds all 16 rows) ----
    const int row_r[2] = {gq, gq + 8};
    int tok_r[2];                                              // new-token index of the lane's two rows
    uint32_t qa[KS][4];
    {
        const uint32_t *qp[2];
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            const int r = row_r[rr];
            tok_r[rr] = r / G;
            const int h = hk * G + r % G;
            qp[rr] = reinterpret_cast<const uint32_t *>(
                (const char *)a.q + (((int64_t)(b.cu_new[s] + min(tok_r[rr], n_s - 1)) * g.Hq + h) * D) * 2);
        }
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
            const int c = ks * 8 + tq;
            qa[ks][0] = row_r[0] < R ? __ldg(qp[0] + c) : 0u;
            qa[ks][1] = row_r[1] < R ? __ldg(qp[1] + c) : 0u;
            qa[ks][2] = row_r[0] < R ? __ldg(qp[0] + c + 4) : 0u;
            qa[ks][3] = row_r[1] < R ? __ldg(qp[1] + c + 4) : 0u;
        }
    }

    float oacc[DB][4];
#pragma unroll
    for (int i = 0; i < DB; ++i) oacc[i][0] = oacc[i][1] = oacc[i][2] = oacc[i][3] = 0.f;
    float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
    const float sl = 1.4426950408889634f * rsqrtf((float)D);      // log2(e)/sqrt(D)

    for (int jt = t_begin; jt < t_end; ++jt) {
        const int st = (jt - t_begin) % kStages;
        asm volatile("cp.async.wait_group %0;" :: "n"(kStages - 2) : "memory");
        __syncthreads();            // tile jt has landed for every thread; every warp is done with tile jt - 1
        {
            const int nx = jt + kStages - 1;                   // goes into the slot tile jt - 1 occupied
            if (nx < t_end) load_tile(nx, (nx - t_begin) % kStages);
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
        const int lb = jt * 4 + w;                             // this warp's pool block of the tile
        if (lb >= nblk_s) continue;                            // no keys in it (warp-uniform)
        const uint32_t ksm = smem_u32(smem + st * kStage) + w * kChunk, vsm = ksm + 4 * kChunk;

        // ---- S = Q K^T : 16 rows x 16 tokens ----
        float sacc[2][4];
#pragma unroll
        for (int i = 0; i < 2; ++i) sacc[i][0] = sacc[i][1] = sacc[i][2] = sacc[i][3] = 0.f;
        {
            const int m = lane >> 3, r = lane & 7;
            const int slot = (m >> 1) * 8 + r;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                uint32_t r0, r1, r2, r3;
                ldsm_x4(ksm + sc_chunk_off(slot, ks * 16 + (m & 1) * 8, NH), r0, r1, r2, r3);
                mma_bf16(sacc[0], qa[ks], r0, r1);
                mma_bf16(sacc[1], qa[ks], r2, r3);
            }
        }
        // ---- causal mask: row r sees keys j <= T_h + r / G ----
        if (lb * 16 + 15 > T_h) {
#pragma unroll
            for (int nb = 0; nb < 2; ++nb)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int j = lb * 16 + nb * 8 + tq * 2 + (e & 1);
                    if (j > T_h + tok_r[e >> 1]) sacc[nb][e] = -INFINITY;
                }
        }
        // ---- online softmax ----
        float alpha[2], msafe[2];
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            float mx = fmaxf(fmaxf(sacc[0][2 * rr], sacc[0][2 * rr + 1]), fmaxf(sacc[1][2 * rr], sacc[1][2 * rr + 1]));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
            const float m_new = fmaxf(m_run[rr], mx);
            msafe[rr] = (m_new == -INFINITY) ? 0.f : m_new;
            alpha[rr] = exp2f((m_run[rr] - msafe[rr]) * sl);
            m_run[rr] = m_new;
        }
        float rs[2] = {0.f, 0.f};
        uint32_t pa[4];
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) {
            float p[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                p[e] = exp2f(sacc[nb][e] * sl - msafe[e >> 1] * sl);
                rs[e >> 1] += p[e];
            }
            pa[nb * 2 + 0] = pack_bf16(p[0], p[1]);
            pa[nb * 2 + 1] = pack_bf16(p[2], p[3]);
        }
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) l_run[rr] = l_run[rr] * alpha[rr] + rs[rr];
        if (alpha[0] != 1.f || alpha[1] != 1.f) {              // the running maximum moved for some row of the lane
#pragma unroll
            for (int i = 0; i < DB; ++i) {
                oacc[i][0] *= alpha[0]; oacc[i][1] *= alpha[0];
                oacc[i][2] *= alpha[1]; oacc[i][3] *= alpha[1];
            }
        }
        // ---- O += P V : 16 rows x 16 tokens x D ----
        {
            const int m = lane >> 3, r = lane & 7;
            const int slot = (m & 1) * 8 + r;
#pragma unroll
            for (int dp = 0; dp < D / 16; ++dp) {
                uint32_t r0, r1, r2, r3;
                ldsm_x4_t(vsm + sc_chunk_off(slot, (dp * 2 + (m >> 1)) * 8, NH), r0, r1, r2, r3);
                mma_bf16(oacc[2 * dp], pa, r0, r1);
                mma_bf16(oacc[2 * dp + 1], pa, r2, r3);
            }
        }
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");

    // ---- merge of the four warps (each holds the rows' state over ITS blocks), then the result ----
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        l_run[rr] += __shfl_xor_sync(0xffffffffu, l_run[rr], 1);
        l_run[rr] += __shfl_xor_sync(0xffffffffu, l_run[rr], 2);
    }
    __syncthreads();                                           // the ring is free
    float *o_w = reinterpret_cast<float *>(smem);              // [4 warps][kRows][D]: each warp's O, rescaled
    float *m_w = o_w + 4 * kRows * D;                          // [4][kRows], log2 units
    float *l_w = m_w + 4 * kRows;                              // [4][kRows]
    if (tq == 0) {
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            m_w[w * kRows + row_r[rr]] = m_run[rr] * sl;       // may be -inf
            l_w[w * kRows + row_r[rr]] = l_run[rr];
        }
    }
    __syncthreads();
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        const int r = row_r[rr];
        if (r >= R) continue;
        const float M = fmaxf(fmaxf(m_w[r], m_w[kRows + r]), fmaxf(m_w[2 * kRows + r], m_w[3 * kRows + r]));
        const float mine = m_run[rr] * sl;
        const float sc = (mine == -INFINITY) ? 0.f : exp2f(mine - M);   // no visible key of the row in this warp's blocks
        float2 *o = reinterpret_cast<float2 *>(o_w + (w * kRows + r) * D);
#pragma unroll
        for (int nb = 0; nb < DB; ++nb) o[nb * 4 + tq] = make_float2(oacc[nb][2 * rr] * sc, oacc[nb][2 * rr + 1] * sc);
    }
    __syncthreads();
    {
        constexpr int CPT = D / 8;                             // values per thread: 8 threads per row
        const int r = tid >> 3, c0 = (tid & 7) * CPT;
        if (r < R) {
            float M = -INFINITY, Lsum = 0.f;
#pragma unroll
            for (int ww = 0; ww < 4; ++ww) M = fmaxf(M, m_w[ww * kRows + r]);
#pragma unroll
            for (int ww = 0; ww < 4; ++ww) {
                const float mw = m_w[ww * kRows + r];
                if (mw != -INFINITY) Lsum += l_w[ww * kRows + r] * exp2f(mw - M);
            }
            const int i = r / G, h = hk * G + r % G;
            const int64_t grow = b.cu_new[s] + i;
            float acc[CPT];                                    // warps added in a fixed order: deterministic
#pragma unroll
            for (int c = 0; c < CPT; ++c)
                acc[c] = (o_w[(0 * kRows + r) * D + c0 + c] + o_w[(1 * kRows + r) * D + c0 + c]) +
                         (o_w[(2 * kRows + r) * D + c0 + c] + o_w[(3 * kRows + r) * D + c0 + c]);
            if (a.n_splits == 1) {
                const float inv = 1.f / Lsum;
                __nv_bfloat16 *o = (__nv_bfloat16 *)a.out + (grow * g.Hq + h) * D + c0;
#pragma unroll
                for (int c = 0; c < CPT; c += 2)
                    *reinterpret_cast<__nv_bfloat162 *>(o + c) = __floats2bfloat162_rn(acc[c] * inv, acc[c + 1] * inv);
            } else {
                const int64_t prow = ((int64_t)split * a.total_new + grow) * g.Hq + h;
                float *o = a.part_o + prow * D + c0;
#pragma unroll
                for (int c = 0; c < CPT; c += 4)
                    *reinterpret_cast<float4 *>(o + c) = make_float4(acc[c], acc[c + 1], acc[c + 2], acc[c + 3]);
                if ((tid & 7) == 0) {
                    a.part_ml[prow * 2 + 0] = M;               // log2 units; -inf if the split holds no visible key
                    a.part_ml[prow * 2 + 1] = Lsum;
                }
            }
        }
    }
}

}  // namespace

int sc_dec_max_rows() { return kRows; }
int sc_dec_split_unit() { return kTileN; }
int sc_dec_ctas_per_sm() { return 2; }

cudaError_t sc_launch_attn_decode(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, cudaStream_t st)
{
    if (a.total_new == 0) return cudaSuccess;
    dim3 grid((unsigned)a.n_splits, (unsigned)g.Hkv, (unsigned)b.n_seq);
    cudaError_t e;
    if (g.D == 128) {
        constexpr int smem = kStages * 8 * 16 * 128 * 2;
        static std::atomic<uint64_t> done{0};
        if (sc_first_use_on_device(done)) {
            e = cudaFuncSetAttribute(sc_attn_decode_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return e;
        }
        sc_attn_decode_kernel<128><<<grid, kThreads, smem, st>>>(g, b, a);
    } else {
        constexpr int smem = kStages * 8 * 16 * 64 * 2;
        static std::atomic<uint64_t> done{0};
        if (sc_first_use_on_device(done)) {
            e = cudaFuncSetAttribute(sc_attn_decode_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return e;
        }
        sc_attn_decode_kernel<64><<<grid, kThreads, smem, st>>>(g, b, a);
    }
    return cudaGetLastError();
}
