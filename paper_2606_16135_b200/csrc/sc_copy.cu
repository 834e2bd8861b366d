// sc_copy.cu -- paged KV movement kernels:
//   scatter : new K/V [n][Hkv][D] -> pool blocks through the table
//   read    : the inverse, pool/LSC -> contiguous [n][Hkv][D] (verification, export)
//   gather  : pool -> LSC, one contiguous cell (Eq. 1 M_block) per logical block
//             ("preloads the KV cache for a given layer into the LSC")
// All of it is byte-exact data movement, bound by HBM (or PCIe for a host pool):
// 16-byte vectors, coalesced, several independent requests in flight per thread; the
// bulk variant moves whole pieces with the TMA engine (cp.async.bulk) through a
// shared-memory ring and keeps the SM's LSU out of it.

#include "sc_internal.h"

namespace {

__device__ __forceinline__ int4 ld_stream(const void *p)
{
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(void *p, const int4 &v)
{
    asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

__device__ __forceinline__ int seq_of(const int32_t *cu, int n_seq, int x)
{
    int s = 0;
    while (s + 1 < n_seq && x >= cu[s + 1]) ++s;
    return s;
}

// ------------------------------------------------------------ scatter / read
// One thread per 16 bytes (8 bf16 of one head of one token, K or V).  The scatter (kToPool) has
// `pad` != 0 when it stores a turn's new tokens: after the n_units data units come, per sequence,
// the 15 slots that may follow its last token inside the last block, and those that exist are
// zero-filled -- slots past the logical end then hold finite values whatever the memory held
// before (attention masks them in S, but 0 * NaN in P.V would poison the row).
template <bool kToPool>
__global__ void __launch_bounds__(256)
sc_scatter_read_kernel(ScGeom g, ScBatch b, char *k_lin, char *v_lin, ScKvView view0,
                       ScKvView view1, int has_view1, int64_t n_units, int pad)
{
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int cpr = g.D >> 3;                       // 16-byte units per head row
    const int c = (int)(idx % cpr);
    int64_t t = idx / cpr;
    const int h = (int)(t % g.Hkv);
    t /= g.Hkv;
    int s, tok, kv;
    int64_t row = 0;
    bool zero = false;
    if (idx < n_units) {
        const int total = b.cu_new[b.n_seq];
        row = t % total;
        kv = (int)(t / total);
        s = seq_of(b.cu_new, b.n_seq, (int)row);
        tok = b.hist[s] + ((int)row - b.cu_new[s]);
    } else {
        if (!kToPool || !pad) return;
        t -= (int64_t)b.cu_new[b.n_seq] * 2;        // (kv, sequence, slot after the end) past the data rows
        const int p = (int)(t % 15);
        t /= 15;
        s = (int)(t % b.n_seq);
        kv = (int)(t / b.n_seq);
        if (kv > 1) return;
        const int end = b.hist[s] + (b.cu_new[s + 1] - b.cu_new[s]);
        if (b.cu_new[s + 1] == b.cu_new[s] || (end & 15) == 0 || (end & 15) + p > 15) return;
        tok = end + p;
        zero = true;
    }
    const int lb = tok >> 4, slot = tok & 15;
    char *lin = (kv ? v_lin : k_lin) + ((row * g.Hkv + h) * g.D + c * 8) * 2;
    const int64_t in_cell = (int64_t)(kv * g.Hkv + h) * g.chunk_bytes + sc_chunk_off(slot, c * 8, g.nh);
    char *p0 = view0.base + sc_phys_block(view0, b, s, lb) * view0.block_stride + in_cell;
    if (kToPool) {
        const int4 val = zero ? make_int4(0, 0, 0, 0) : ld_stream(lin);
        *reinterpret_cast<int4 *>(p0) = val;
        if (has_view1) {
            char *p1 = view1.base + sc_phys_block(view1, b, s, lb) * view1.block_stride + in_cell;
            *reinterpret_cast<int4 *>(p1) = val;
        }
    } else {
        *reinterpret_cast<int4 *>(lin) = *reinterpret_cast<const int4 *>(p0);
    }
}

// ------------------------------------------------------------ gather (LDG/STG)
constexpr int kGatherThreads = 128;   // small CTAs: one fits beside a tcgen05 attention CTA (registers)
constexpr int kGatherUnroll = 8;
constexpr int kGatherPiece = kGatherThreads * 16 * kGatherUnroll;   // 16 KiB per CTA

__global__ void __launch_bounds__(kGatherThreads)
sc_gather_ldg_kernel(ScGeom g, ScBatch b, ScKvView src, ScKvView dst, int pieces_per_cell)
{
    const int gb = blockIdx.x / pieces_per_cell;
    const int piece = blockIdx.x - gb * pieces_per_cell;
    const int s = seq_of(b.cu_blk, b.n_seq, gb);
    const int j = gb - b.cu_blk[s] + b.rc_blk[s];          // resident blocks are not gathered
    const char *sp = src.base + sc_phys_block(src, b, s, j) * src.block_stride;
    char *dp = dst.base + sc_phys_block(dst, b, s, j) * dst.block_stride;
    const int64_t off0 = (int64_t)piece * kGatherPiece + threadIdx.x * 16;
    // pool lines are read once per layer: evict them first, so that the LSC lines this kernel writes
    // (and the next layer's attention reads) have a better chance of still being in L2 by then.
    // (Measured with the attention's LSC reads marked the same way: staged lwm_5k turn 1.86 -> 1.79 ms;
    // an evict_last policy on the stores below changed nothing.)
    uint64_t pol_rd;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_rd));
    int4 v[kGatherUnroll];
#pragma unroll
    for (int u = 0; u < kGatherUnroll; ++u) {
        const int64_t off = off0 + (int64_t)u * kGatherThreads * 16;
        if (off < g.cell_bytes)
            asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.v4.s32 {%0,%1,%2,%3}, [%4], %5;"
                         : "=r"(v[u].x), "=r"(v[u].y), "=r"(v[u].z), "=r"(v[u].w) : "l"(sp + off), "l"(pol_rd));
    }
#pragma unroll
    for (int u = 0; u < kGatherUnroll; ++u) {
        const int64_t off = off0 + (int64_t)u * kGatherThreads * 16;
        if (off < g.cell_bytes) *reinterpret_cast<int4 *>(dp + off) = v[u];
    }
}

// ------------------------------------------------------------ gather (TMA bulk)
// One thread per CTA drives a ring of kBulkStages pieces: cp.async.bulk global->shared
// completing on an mbarrier, then cp.async.bulk shared->global in a bulk group.
constexpr int kBulkStages = 6;
constexpr int kBulkPiece = 32 * 1024;

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;"
                 :: "r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// bounded like the attention kernel's waits: after ~2 s of failed probes the kernel traps instead of
// hanging the GPU on a protocol error
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    uint32_t ok;
    long long t0 = 0;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
        if (ok) return;
        const long long t = clock64();
        if (t0 == 0) t0 = t;
        else if (t - t0 > 4000000000ll) __trap();
    }
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        :: "r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *gdst, const void *smem_src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 :: "l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}

__global__ void __launch_bounds__(32)
sc_gather_bulk_kernel(ScGeom g, ScBatch b, ScKvView src, ScKvView dst, int pieces_per_cell,
                      int piece_bytes, int n_items)
{
    extern __shared__ __align__(128) char ring[];
    __shared__ uint64_t full[kBulkStages];
    if (threadIdx.x != 0) return;
    for (int i = 0; i < kBulkStages; ++i) mbar_init(&full[i], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");

    // this CTA's items: blockIdx.x, blockIdx.x + gridDim.x, ...
    const int my_n = (n_items - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    auto locate = [&](int it, const char *&sp, char *&dp) {
        const int item = blockIdx.x + it * gridDim.x;
        const int gb = item / pieces_per_cell, piece = item - gb * pieces_per_cell;
        const int s = seq_of(b.cu_blk, b.n_seq, gb);
        const int j = gb - b.cu_blk[s] + b.rc_blk[s];      // resident blocks are not gathered
        const int64_t off = (int64_t)piece * piece_bytes;
        sp = src.base + sc_phys_block(src, b, s, j) * src.block_stride + off;
        dp = dst.base + sc_phys_block(dst, b, s, j) * dst.block_stride + off;
    };
    auto issue_load = [&](int it) {
        const char *sp; char *dp;
        locate(it, sp, dp);
        const int st = it % kBulkStages;
        mbar_expect_tx(&full[st], (uint32_t)piece_bytes);
        bulk_g2s(ring + (size_t)st * kBulkPiece, sp, (uint32_t)piece_bytes, &full[st]);
    };
    const int pro = my_n < kBulkStages ? my_n : kBulkStages;
    for (int it = 0; it < pro; ++it) issue_load(it);
    for (int it = 0; it < my_n; ++it) {
        const int st = it % kBulkStages;
        mbar_wait(&full[st], (uint32_t)((it / kBulkStages) & 1));
        const char *sp; char *dp;
        locate(it, sp, dp);
        bulk_s2g(dp, ring + (size_t)st * kBulkPiece, (uint32_t)piece_bytes);
        if (it >= 1 && it - 1 + kBulkStages < my_n) {
            // the store of item it-1 must have finished READING its stage before refill
            asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
            issue_load(it - 1 + kBulkStages);
        }
    }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

}  // namespace

// ------------------------------------------------------------------ launchers
cudaError_t sc_launch_scatter(const ScGeom &g, const void *k, const void *v, const ScBatch &b,
                              const ScKvView &dst0, const ScKvView *dst1, bool pad_last_block, cudaStream_t st)
{
    const int64_t per_row = (int64_t)g.Hkv * (g.D / 8);
    const int64_t units = (int64_t)b.cu_new[b.n_seq] * 2 * per_row;
    if (units == 0) return cudaSuccess;
    const int64_t pad_units = pad_last_block ? (int64_t)b.n_seq * 2 * 15 * per_row : 0;
    const unsigned grid = (unsigned)((units + pad_units + 255) / 256);
    sc_scatter_read_kernel<true><<<grid, 256, 0, st>>>(g, b, (char *)k, (char *)v, dst0,
                                                        dst1 ? *dst1 : dst0, dst1 != nullptr, units, pad_last_block);
    return cudaGetLastError();
}

cudaError_t sc_launch_read(const ScGeom &g, void *k_out, void *v_out, const ScBatch &b,
                           const ScKvView &src, cudaStream_t st)
{
    const int64_t units = (int64_t)b.cu_new[b.n_seq] * 2 * g.Hkv * (g.D / 8);
    if (units == 0) return cudaSuccess;
    const unsigned grid = (unsigned)((units + 255) / 256);
    sc_scatter_read_kernel<false><<<grid, 256, 0, st>>>(g, b, (char *)k_out, (char *)v_out, src, src,
                                                         0, units, 0);
    return cudaGetLastError();
}

cudaError_t sc_launch_gather(const ScGeom &g, const ScBatch &b, const ScKvView &src,
                             const ScKvView &dst, int engine, int n_sms, cudaStream_t st)
{
    const int total_blocks = b.cu_blk[b.n_seq];
    if (total_blocks == 0) return cudaSuccess;
    if (engine == SC_COPY_BULK) {
        const int piece = g.cell_bytes < kBulkPiece ? (int)g.cell_bytes : kBulkPiece;
        const int ppc = (int)(g.cell_bytes / piece);     // cell_bytes is a multiple of 4 KiB
        if ((int64_t)ppc * piece == g.cell_bytes) {
            const int n_items = total_blocks * ppc;
            static std::atomic<uint64_t> done{0};
            const int smem = kBulkStages * kBulkPiece;
            if (sc_first_use_on_device(done)) {
                cudaError_t e = cudaFuncSetAttribute(sc_gather_bulk_kernel,
                                                     cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
                if (e != cudaSuccess) return e;
            }
            const int grid = n_sms < n_items ? n_sms : n_items;
            sc_gather_bulk_kernel<<<grid, 32, smem, st>>>(g, b, src, dst, ppc, piece, n_items);
            return cudaGetLastError();
        }
        // odd cell size: fall through to the vector copy
    }
    const int ppc = (int)((g.cell_bytes + kGatherPiece - 1) / kGatherPiece);
    sc_gather_ldg_kernel<<<(unsigned)(total_blocks * ppc), kGatherThreads, 0, st>>>(g, b, src, dst, ppc);
    return cudaGetLastError();
}
