// sc_attn_mma.cu -- paged prefill attention, mma.sync engine, and the split-KV combine
// (each new token attends to all history
// tokens and to the new tokens up to and including itself).
//
// This is the first, register-accumulator engine: flash-style online softmax over
// 64-token KV tiles fetched through the block table with cp.async (one contiguous
// chunk per (block, head)), QK^T and PV on mma.sync.m16n8k16 bf16 with fp32
// accumulation.  The tcgen05/TMEM engine lives in sc_attn_tc.cu; both produce
// partial (m, l, O) triples merged by sc_combine_kernel when the keys are split
// across CTAs.  Work partitioning depends on logical positions only, so results are
// bit-identical under any permutation of physical block ids.
#include <cuda_bf16.h>

#include "sc_internal.h"

namespace {

constexpr int kTileM = 64;    // query rows per CTA (16 per warp)
constexpr int kTileN = 64;    // KV tokens per tile (4 pool blocks)
constexpr int kThreads = 128;

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
__device__ __forceinline__ int seq_of(const int32_t *cu, int n_seq, int x)
{
    int s = 0;
    while (s + 1 < n_seq && x >= cu[s + 1]) ++s;
    return s;
}

template <int D>
__global__ void __launch_bounds__(kThreads)
sc_attn_mma_kernel(ScGeom g, ScBatch b, ScAttnArgs a)
{
    constexpr int kChunk = 16 * D * 2;            // bytes of one (block, head) chunk
    constexpr int kStage = 8 * kChunk;            // K: 4 chunks, V: 4 chunks
    constexpr int NH = D / 64;
    constexpr int KS = D / 16;                    // k-steps of QK^T
    constexpr int NB = kTileN / 8;                // 8 n-blocks of S
    constexpr int DB = D / 8;                     // n-blocks of O
    extern __shared__ __align__(1024) char smem[];

    const int split = blockIdx.x, h = blockIdx.y, gmt = blockIdx.z;
    const int s = seq_of(b.cu_mt, b.n_seq, gmt);
    const int mt = gmt - b.cu_mt[s];
    const int n_s = b.cu_new[s + 1] - b.cu_new[s];
    const int T_h = b.hist[s];
    const int i0 = mt * kTileM;
    const int rows_valid = min(kTileM, n_s - i0);
    const int kmax = T_h + i0 + rows_valid;                 // keys [0, kmax) are visible to the tile
    const int tiles_needed = (kmax + kTileN - 1) / kTileN;
    const int t_begin = split * a.split_units;
    const int t_end = min(t_begin + a.split_units, tiles_needed);
    if (t_begin >= t_end) return;
    const int nblk_s = (T_h + n_s + 15) >> 4;
    const int hk = h / (g.Hq / g.Hkv);
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    const int gq = lane >> 2, tq = lane & 3;

    // ---- Q fragments straight from global (once per CTA) ----
    uint32_t qa[KS][4];
    {
        const int r0 = i0 + w * 16 + gq, r1 = r0 + 8;
        const uint32_t *q0 = reinterpret_cast<const uint32_t *>(
            (const char *)a.q + (((int64_t)(b.cu_new[s] + r0) * g.Hq + h) * D) * 2);
        const uint32_t *q1 = reinterpret_cast<const uint32_t *>(
            (const char *)a.q + (((int64_t)(b.cu_new[s] + r1) * g.Hq + h) * D) * 2);
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
            const int c = ks * 8 + tq;              // uint32 index = (ks*16 + tq*2)/2
            qa[ks][0] = r0 < n_s ? __ldg(q0 + c) : 0u;
            qa[ks][1] = r1 < n_s ? __ldg(q1 + c) : 0u;
            qa[ks][2] = r0 < n_s ? __ldg(q0 + c + 4) : 0u;
            qa[ks][3] = r1 < n_s ? __ldg(q1 + c + 4) : 0u;
        }
    }

    auto load_tile = [&](int jt, int st) {
        char *dst = smem + st * kStage;
#pragma unroll
        for (int ci = 0; ci < 8; ++ci) {
            const int kvsel = ci >> 2, blk = ci & 3;
            const int lb = min(jt * 4 + blk, nblk_s - 1);
            const char *src = a.kv.base + sc_phys_block(a.kv, b, s, lb) * a.kv.block_stride +
                              (int64_t)(kvsel * g.Hkv + hk) * kChunk;
#pragma unroll
            for (int off = tid * 16; off < kChunk; off += kThreads * 16)
                cp_async16(smem_u32(dst + ci * kChunk + off), src + off);
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    float oacc[DB][4];
#pragma unroll
    for (int i = 0; i < DB; ++i) oacc[i][0] = oacc[i][1] = oacc[i][2] = oacc[i][3] = 0.f;
    float m_run[2] = {-INFINITY, -INFINITY}, l_run[2] = {0.f, 0.f};
    const float sl = 1.4426950408889634f * rsqrtf((float)D);      // log2(e)/sqrt(D)
    const int row_l[2] = {i0 + w * 16 + gq, i0 + w * 16 + gq + 8};

    load_tile(t_begin, 0);
    for (int jt = t_begin; jt < t_end; ++jt) {
        const int st = (jt - t_begin) & 1;
        if (jt + 1 < t_end) {
            load_tile(jt + 1, st ^ 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncthreads();
        const uint32_t ksm = smem_u32(smem + st * kStage), vsm = ksm + 4 * kChunk;

        // ---- S = Q K^T ----
        float sacc[NB][4];
#pragma unroll
        for (int i = 0; i < NB; ++i) sacc[i][0] = sacc[i][1] = sacc[i][2] = sacc[i][3] = 0.f;
        {
            const int m = lane >> 3, r = lane & 7;
            const int slot = (m >> 1) * 8 + r;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                const uint32_t coff = sc_chunk_off(slot, ks * 16 + (m & 1) * 8, NH);
#pragma unroll
                for (int np = 0; np < 4; ++np) {
                    uint32_t r0, r1, r2, r3;
                    ldsm_x4(ksm + np * kChunk + coff, r0, r1, r2, r3);
                    mma_bf16(sacc[2 * np], qa[ks], r0, r1);
                    mma_bf16(sacc[2 * np + 1], qa[ks], r2, r3);
                }
            }
        }
        // ---- causal mask (only tiles that reach past the first row's limit) ----
        if (jt * kTileN + kTileN - 1 > T_h + i0 + w * 16) {
#pragma unroll
            for (int nb = 0; nb < NB; ++nb)
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int j = jt * kTileN + nb * 8 + tq * 2 + (e & 1);
                    if (j > T_h + row_l[e >> 1]) sacc[nb][e] = -INFINITY;
                }
        }
        // ---- online softmax ----
        float alpha[2], msafe[2];
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) {
            float mx = -INFINITY;
#pragma unroll
            for (int nb = 0; nb < NB; ++nb) mx = fmaxf(mx, fmaxf(sacc[nb][2 * rr], sacc[nb][2 * rr + 1]));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
            const float m_new = fmaxf(m_run[rr], mx);
            msafe[rr] = (m_new == -INFINITY) ? 0.f : m_new;
            alpha[rr] = exp2f((m_run[rr] - msafe[rr]) * sl);
            m_run[rr] = m_new;
        }
        float rs[2] = {0.f, 0.f};
        uint32_t pa[4][4];
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
            float p[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                p[e] = exp2f(sacc[nb][e] * sl - msafe[e >> 1] * sl);
                rs[e >> 1] += p[e];
            }
            pa[nb >> 1][(nb & 1) * 2 + 0] = pack_bf16(p[0], p[1]);
            pa[nb >> 1][(nb & 1) * 2 + 1] = pack_bf16(p[2], p[3]);
        }
#pragma unroll
        for (int rr = 0; rr < 2; ++rr) l_run[rr] = l_run[rr] * alpha[rr] + rs[rr];
#pragma unroll
        for (int i = 0; i < DB; ++i) {
            oacc[i][0] *= alpha[0]; oacc[i][1] *= alpha[0];
            oacc[i][2] *= alpha[1]; oacc[i][3] *= alpha[1];
        }
        // ---- O += P V ----
        {
            const int m = lane >> 3, r = lane & 7;
            const int slot = (m & 1) * 8 + r;
#pragma unroll
            for (int kt = 0; kt < 4; ++kt) {
#pragma unroll
                for (int dp = 0; dp < D / 16; ++dp) {
                    const uint32_t coff = sc_chunk_off(slot, (dp * 2 + (m >> 1)) * 8, NH);
                    uint32_t r0, r1, r2, r3;
                    ldsm_x4_t(vsm + kt * kChunk + coff, r0, r1, r2, r3);
                    mma_bf16(oacc[2 * dp], pa[kt], r0, r1);
                    mma_bf16(oacc[2 * dp + 1], pa[kt], r2, r3);
                }
            }
        }
        __syncthreads();
    }

    // ---- epilogue ----
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        l_run[rr] += __shfl_xor_sync(0xffffffffu, l_run[rr], 1);
        l_run[rr] += __shfl_xor_sync(0xffffffffu, l_run[rr], 2);
    }
#pragma unroll
    for (int rr = 0; rr < 2; ++rr) {
        const int i = row_l[rr];
        if (i >= n_s) continue;
        const int64_t grow = b.cu_new[s] + i;
        if (a.n_splits == 1) {
            const float inv = 1.f / l_run[rr];
            uint32_t *o = reinterpret_cast<uint32_t *>((char *)a.out + ((grow * g.Hq + h) * D) * 2);
#pragma unroll
            for (int nb = 0; nb < DB; ++nb)
                o[nb * 4 + tq] = pack_bf16(oacc[nb][2 * rr] * inv, oacc[nb][2 * rr + 1] * inv);
        } else {
            const int64_t prow = ((int64_t)split * a.total_new + grow) * g.Hq + h;
            float2 *o = reinterpret_cast<float2 *>(a.part_o + prow * D);
#pragma unroll
            for (int nb = 0; nb < DB; ++nb)
                o[nb * 4 + tq] = make_float2(oacc[nb][2 * rr], oacc[nb][2 * rr + 1]);
            if (tq == 0) {
                a.part_ml[prow * 2 + 0] = m_run[rr] * sl;      // log2 units; may be -inf
                a.part_ml[prow * 2 + 1] = l_run[rr];
            }
        }
    }
}

// ------------------------------------------------------------------ combine (a7)
// One warp per (row, head): O = sum_s 2^(m_s-M) O_s / sum_s 2^(m_s-M) l_s, splits in order.
// HALF: the partial rows are fp16 scaled by a power of two (the tcgen05 engine: m carries the exponent,
// l the scaled sum), else fp32 (the mma.sync engine).  Lane sp holds (m, l) of split sp; the O rows of
// four splits are requested before the first is used.
template <int D, bool HALF>
__global__ void __launch_bounds__(256)
sc_combine_kernel(ScGeom g, ScBatch b, ScAttnArgs a, int tile_m, int split_unit)
{
    const int64_t wid = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wid >= (int64_t)a.total_new * g.Hq) return;
    const int h = (int)(wid % g.Hq);
    const int grow = (int)(wid / g.Hq);
    const int s = seq_of(b.cu_new, b.n_seq, grow);
    const int i = grow - b.cu_new[s];
    const int n_s = b.cu_new[s + 1] - b.cu_new[s];
    const int mt = i / tile_m;
    const int rows_valid = min(tile_m, n_s - mt * tile_m);
    const int kmax = b.hist[s] + mt * tile_m + rows_valid;
    const int units_needed = (kmax + split_unit - 1) / split_unit;
    const int ns = (units_needed + a.split_units - 1) / a.split_units;      // <= 32 (max_splits)
    constexpr int V = D / 32;                                  // values per lane
    auto prow_of = [&](int sp) { return ((int64_t)sp * a.total_new + grow) * g.Hq + h; };
    float my_m = -INFINITY, my_l = 0.f;
    if (lane < ns) {
        const float2 ml = *reinterpret_cast<const float2 *>(a.part_ml + prow_of(lane) * 2);
        my_m = ml.x; my_l = ml.y;
    }
    float M = my_m;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, o));
    const float my_w = (my_m == -INFINITY) ? 0.f : exp2f(my_m - M);
    float acc[V];
#pragma unroll
    for (int v = 0; v < V; ++v) acc[v] = 0.f;
    float W = 0.f;
    for (int sp0 = 0; sp0 < ns; sp0 += 4) {
        float o[4][V];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int sp = min(sp0 + q, ns - 1);
            const float wq = __shfl_sync(0xffffffffu, my_w, sp);
#pragma unroll
            for (int v = 0; v < V; ++v) o[q][v] = 0.f;
            if (sp0 + q < ns && wq != 0.f) {          // O_s of a split of weight 0 may never have been written
                if (HALF) {
                    const __half *p = reinterpret_cast<const __half *>(a.part_o) + prow_of(sp) * D + lane * V;
#pragma unroll
                    for (int v = 0; v < V; v += 2) {
                        const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(p + v));
                        o[q][v] = f.x; o[q][v + 1] = f.y;
                    }
                } else {
                    const float *p = a.part_o + prow_of(sp) * D + lane * V;
#pragma unroll
                    for (int v = 0; v < V; ++v) o[q][v] = p[v];
                }
            }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int sp = sp0 + q;
            const float wq = __shfl_sync(0xffffffffu, my_w, min(sp, ns - 1)), lq = __shfl_sync(0xffffffffu, my_l, min(sp, ns - 1));
            if (sp < ns && wq != 0.f) {
                W += wq * lq;
#pragma unroll
                for (int v = 0; v < V; ++v) acc[v] += wq * o[q][v];
            }
        }
    }
    const float inv = 1.f / W;
    __nv_bfloat16 *out = (__nv_bfloat16 *)a.out + ((int64_t)grow * g.Hq + h) * D + lane * V;
#pragma unroll
    for (int v = 0; v < V; v += 2)
        *reinterpret_cast<__nv_bfloat162 *>(out + v) = __floats2bfloat162_rn(acc[v] * inv, acc[v + 1] * inv);
}

}  // namespace

int sc_mma_tile_m() { return kTileM; }
int sc_mma_split_unit() { return kTileN; }

cudaError_t sc_launch_attn_mma(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, cudaStream_t st)
{
    const int total_mt = b.cu_mt[b.n_seq];
    if (total_mt == 0) return cudaSuccess;
    dim3 grid((unsigned)a.n_splits, (unsigned)g.Hq, (unsigned)total_mt);
    cudaError_t e;
    if (g.D == 128) {
        constexpr int smem = 2 * 8 * 16 * 128 * 2;
        static std::atomic<uint64_t> done{0};
        if (sc_first_use_on_device(done)) {
            e = cudaFuncSetAttribute(sc_attn_mma_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return e;
        }
        sc_attn_mma_kernel<128><<<grid, kThreads, smem, st>>>(g, b, a);
    } else {
        constexpr int smem = 2 * 8 * 16 * 64 * 2;
        sc_attn_mma_kernel<64><<<grid, kThreads, smem, st>>>(g, b, a);
    }
    return cudaGetLastError();
}

cudaError_t sc_launch_combine(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, int tile_m,
                              int split_unit, cudaStream_t st)
{
    const int64_t warps = (int64_t)a.total_new * g.Hq;
    if (warps == 0) return cudaSuccess;
    const unsigned grid = (unsigned)((warps * 32 + 255) / 256);
    if (a.part_half) {
        if (g.D == 128) sc_combine_kernel<128, true><<<grid, 256, 0, st>>>(g, b, a, tile_m, split_unit);
        else sc_combine_kernel<64, true><<<grid, 256, 0, st>>>(g, b, a, tile_m, split_unit);
    } else {
        if (g.D == 128) sc_combine_kernel<128, false><<<grid, 256, 0, st>>>(g, b, a, tile_m, split_unit);
        else sc_combine_kernel<64, false><<<grid, 256, 0, st>>>(g, b, a, tile_m, split_unit);
    }
    return cudaGetLastError();
}
