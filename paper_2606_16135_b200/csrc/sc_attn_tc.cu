// sc_attn_tc.cu -- paged prefill attention, tcgen05 / TMEM engine (
// each new token attends to all history tokens and to the new tokens up to
// and including itself).
//
// One CTA owns a PAIR of 128-row query tiles of one query head (256 new tokens) and a
// contiguous range of 16-token pool blocks (one split), walked in KV tiles of 8 blocks; the
// last tile of a split may hold fewer blocks (the MMAs then use N = 16 * blocks).  Warp roles:
//   warp 0      producer : per KV tile, up to 8 + 8 bulk copies (cp.async.bulk, 4 KiB each)
//                          bring the K and V chunks of the tile's pool blocks -- found through
//                          the block table -- into a 5-slot shared-memory ring.  The pool
//                          stores chunks in the tensor core's 128B-swizzled operand order
//                          (include/swiftcache.h), so a chunk is an MMA operand as it lands.
//   warp 1      MMA      : one thread issues tcgen05.mma.  S_m = Q_m K^T (both operands in
//                          shared memory, K-major) into TMEM; O_m += P_m V with P_m read from
//                          TMEM and V as an MN-major shared-memory operand.
//   warp 2      TMEM allocation (all 512 columns: S0 S1 O0 O1, 128 fp32 columns each);
//   warps 2-3   in cluster mode: this CTA's share of the scatter of the new K/V (a5)
//   warps 4-7   softmax warpgroup of query tile 0: thread r owns row r.  S is read from TMEM
//   warps 8-11  same for query tile 1            : 32 columns at a time, online softmax in
//                          registers against a LAZY reference maximum (advanced, and O
//                          rescaled, only when the row max grows by > 2^8), P rounded to bf16
//                          and stored over S in TMEM, epilogue.
// The two query tiles ping-pong on the tensor pipe: while warpgroup 0 does the softmax of
// tile j, the pipe runs PV and QK^T of query tile 1.
//
// Split-KV (a7): with up to 16 splits that fit one wave, the CTAs of one (query pair, head) are
// a thread-block cluster; they share the scatter and merge their partial (m, l, O) through
// distributed shared memory at the end (row-scaled fp16 partials moved by the TMA engine).
// Otherwise partials go to global scratch and sc_combine_kernel merges them, and the scatter
// kernel runs before this one.
//
// Work partitioning depends on logical positions only, so results are bit-identical under
// any permutation of physical block ids, and staged attention is this same kernel run with
// the identity table over the LSC.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include <type_traits>

#include "sc_internal.h"

namespace {

constexpr int kTM = 128;          // rows of one query tile
constexpr int kPairM = 2 * kTM;   // rows a CTA owns
constexpr int kTN = 128;          // KV tokens per full tile (8 pool blocks)
constexpr int kTileBlks = 8;
constexpr int kStages = 5;        // ring slots (each holds the K or the V half of a tile)
constexpr int kThreads = 384;
constexpr int kMaxCluster = 16;   // most splits merged in kernel (non-portable cluster size)
constexpr float kRescaleThreshold = 8.f;   // log2 units
// Registers.  LEAN = 1 (staged mode): launched with 152 per thread, not the 168 that 384
// threads could have, so that a 128-thread gather CTA of the copy stream fits beside an
// attention CTA on the same SM; warps 0-3 then shrink to 56 and the softmax warps grow to 200
// (setmaxnreg).  LEAN = 0 (fused mode, nothing to share the SM with): 168 -> 72 / 208.
// Either way 384 threads x >= 152 registers leave room for only ONE attention CTA per SM, also at
// D = 64 where two would fit in shared memory: each CTA allocates all 512 TMEM columns, and two
// CTAs of one cluster on the same SM would wait for each other (TMEM vs cluster barrier).

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return (uint32_t)__cvta_generic_to_shared(p);
}

// ------------------------------------------------------------------ mbarrier
__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
// A wait that cannot hang the GPU: after ~2 s of failed probes the kernel traps (surfaces as
// SC_ERR_CUDA on the next call) instead of spinning forever on a protocol error.  Each probe
// carries a suspend-time hint: the thread sleeps in hardware until the phase completes (or the
// hint runs out) instead of polling -- a polling warp takes issue slots from the softmax warp
// that shares its scheduler.
constexpr uint32_t kSuspendNs = 200000;
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    long long t0 = 0;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity), "r"(kSuspendNs) : "memory");
        if (ok) return;
        const long long t = clock64();
        if (t0 == 0) t0 = t;
        else if (t - t0 > 4000000000ll) __trap();
    }
}
// same, acquiring at cluster scope (the arrivals / bytes come from other CTAs of the cluster)
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    long long t0 = 0;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity), "r"(kSuspendNs) : "memory");
        if (ok) return;
        const long long t = clock64();
        if (t0 == 0) t0 = t;
        else if (t - t0 > 4000000000ll) __trap();
    }
}
__device__ __forceinline__ void bulk_g2s(uint32_t smem_dst, const void *gsrc, uint32_t bytes, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        :: "r"(smem_dst), "l"(gsrc), "r"(bytes), "r"(bar) : "memory");
}
// the same with an L2 cache policy (createpolicy) for the lines it touches
__device__ __forceinline__ void bulk_g2s_hint(uint32_t smem_dst, const void *gsrc, uint32_t bytes, uint32_t bar, uint64_t pol)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        :: "r"(smem_dst), "l"(gsrc), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
// this CTA's shared memory -> a peer CTA's shared memory (destination and barrier are addresses
// in the shared::cluster window of the peer), completing on the PEER's mbarrier
__device__ __forceinline__ void bulk_s2peer(uint32_t peer_dst, uint32_t src, uint32_t bytes, uint32_t peer_bar)
{
    asm volatile(
        "cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
        :: "r"(peer_dst), "r"(src), "r"(bytes), "r"(peer_bar) : "memory");
}
__device__ __forceinline__ uint32_t mapa(uint32_t addr, int cta)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(cta));
    return r;
}

// all threads of all CTAs of the cluster; release / acquire at cluster scope (global writes included)
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_sync_all() { cluster_arrive(); cluster_wait(); }

// ------------------------------------------------------------------ tcgen05
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// shared-memory matrix descriptor, 128-byte swizzle, version 1 (Blackwell)
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor: bf16 x bf16 -> fp32, M = 128, A K-major
__host__ __device__ constexpr uint32_t make_idesc(int n, int b_mn_major)
{
    return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)b_mn_major << 16) | ((uint32_t)(n >> 3) << 17) |
           ((uint32_t)(kTM >> 4) << 24);
}
__device__ __forceinline__ void umma_ss(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        :: "r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void umma_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}"
        :: "r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(acc) : "memory");
}
// arrives on `bar` when every tcgen05.mma issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}

// 32 lanes x 32 columns of 32-bit: thread i of the warp gets lane (base + i), columns col..col+31
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%32], "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31};"
        :: "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]),
           "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]),
           "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]),
           "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]),
           "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// tcgen05.wait::ld naming the registers the load is still writing as in/out operands: nothing
// that reads them can be scheduled above the wait.
__device__ __forceinline__ void tmem_ld_wait(uint32_t (&r)[32])
{
    asm volatile(
        "tcgen05.wait::ld.sync.aligned;"
        : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
          "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15]),
          "+r"(r[16]), "+r"(r[17]), "+r"(r[18]), "+r"(r[19]), "+r"(r[20]), "+r"(r[21]), "+r"(r[22]), "+r"(r[23]),
          "+r"(r[24]), "+r"(r[25]), "+r"(r[26]), "+r"(r[27]), "+r"(r[28]), "+r"(r[29]), "+r"(r[30]), "+r"(r[31])
        :: "memory");
}
// 32 lanes x 16 columns (the pipelined softmax reads S in pieces of 16 columns)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait(uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.wait::ld.sync.aligned;"
        : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
          "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])
        :: "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// ---- packed fp32x2 arithmetic (FFMA2 / FADD2 on sm_100): halves the FMA-pipe instructions of the softmax ----
__device__ __forceinline__ uint64_t pk2(float lo, float hi)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(uint64_t v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ uint64_t fma2(uint64_t a, uint64_t b, uint64_t c)
{
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ uint64_t add2(uint64_t a, uint64_t b)
{
    uint64_t d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ float max3(float a, float b, float c)      // FMNMX3 on sm_100
{
    float d;
    asm("max.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c));
    return d;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&v);
}
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi)
{
    __half2 v = __floats2half2_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&v);
}
__device__ __forceinline__ float2 unpack_f16(uint32_t u)
{
    return __half22float2(*reinterpret_cast<__half2 *>(&u));
}
__device__ __forceinline__ int seq_of(const int32_t *cu, int n_seq, int x)
{
    int s = 0;
    while (s + 1 < n_seq && x >= cu[s + 1]) ++s;
    return s;
}

// shared-memory plan (offsets from the 1024-byte aligned base)
//   [kQOff]     Q_0, Q_1 (swizzled like K tiles); in the cluster epilogue: this CTA's partial O, one
//               row-scaled fp16 row of D values per query row, 16-byte units XORed with the row index
//   [kRingOff]  the KV ring; in the cluster epilogue: what the peers send, [split][row][D] fp16 and,
//               from kRecvMlOff, [split][row] (A, L); from kMlOff this CTA's own (A, L) per query row
//               (written only after BOTH query tiles' last MMA: until then the ring is in use)
//   [kBarOff]   mbarriers, TMEM base
// The total stays 1 KiB under the per-SM limit so that a gather CTA of the copy stream (no shared memory
// of its own, but 1 KiB is reserved per resident CTA) still fits beside an attention CTA in staged mode.
template <int D>
struct Plan {
    static constexpr int NH = D / 64;
    static constexpr int kChunk = 16 * D * 2;          // one (block, head) chunk
    static constexpr int kQTile = kTM * D * 2;         // one query tile, swizzled like a K tile
    static constexpr int kSlot = kTN * D * 2;          // K (or V) of one KV tile = 8 chunks
    static constexpr int kRowB = D * 2;                // one fp16 row of a partial O
    static constexpr int kRecvRows = kPairM + 2 * kMaxCluster;   // rows_per_cta (even) * splits <= this
    static constexpr int kQOff = 0;
    static constexpr int kRingOff = 2 * kQTile;
    static constexpr int kRecvMlOff = kRecvRows * kRowB;          // inside the ring
    static constexpr int kMlOff = kRingOff + kRecvMlOff + kRecvRows * 8;
    static constexpr int kBarOff = kRingOff + kStages * kSlot;
    static constexpr int kSlack = 832;                 // the dynamic window may start this far off a 1 KiB boundary
    static constexpr int kBytes = kBarOff + 192 + kSlack;
    static_assert(kMlOff + kPairM * 8 <= kBarOff, "receive and staging areas must fit in the ring");
    static_assert(kBytes <= 232448 - 1024, "no room left for a co-resident gather CTA");
};

struct Bars {                       // at Plan::kBarOff
    uint64_t full[kStages], empty[kStages];
    uint64_t s_ready[2];            // MMA -> softmax warpgroup m: S_m written (and earlier PV_m done)
    uint64_t p_ready[2];            // softmax warpgroup m -> MMA: P_m stored, O_m rescaled
    uint64_t q_ready[2];            // Q_m in shared memory
    uint64_t q_stage[2];            // the rows of Q_m have landed in their staging slot
    uint64_t scat_done;             // warps 2-3 -> producer: this CTA's share of the new K/V is in the pool
    uint64_t recv;                  // cluster epilogue: the peers' partials have landed in this CTA
    uint32_t tmem_base;
};
static_assert(sizeof(Bars) <= 192, "Bars outgrew its slot");

template <int D, int LEAN>
__global__ void __maxnreg__(LEAN ? 152 : 168)
sc_attn_tc_kernel(ScGeom g, ScBatch b, ScAttnArgs a)
{
    using P = Plan<D>;
    constexpr int NH = P::NH;
    extern __shared__ char smem_raw[];
    const uint32_t raw_u32 = smem_u32(smem_raw);
    const uint32_t base = (raw_u32 + 1023u) & ~1023u;
    if (base - raw_u32 > (uint32_t)P::kSlack) __trap();          // never seen: the window starts on a 1 KiB boundary
    char *smem = smem_raw + (base - raw_u32);
    Bars *bars = reinterpret_cast<Bars *>(smem + P::kBarOff);

    // ---- which work is this CTA's (all of it warp- and CTA-uniform) ----
    const int split = blockIdx.x, h = blockIdx.y, gp = blockIdx.z;
    const int s = seq_of(b.cu_mt, b.n_seq, gp);
    const int pair = gp - b.cu_mt[s];
    const int n_s = b.cu_new[s + 1] - b.cu_new[s];
    const int T_h = b.hist[s];
    const int tok0 = pair * kPairM;
    int rows[2], need[2], nt[2];                 // need: pool blocks query tile m can see
#pragma unroll
    for (int m = 0; m < 2; ++m) {
        rows[m] = max(0, min(kTM, n_s - tok0 - m * kTM));
        need[m] = rows[m] > 0 ? (T_h + tok0 + m * kTM + rows[m] + 15) >> 4 : 0;
    }
    const int need_max = max(need[0], need[1]);
    const int b_begin = split * a.split_units;   // this split's blocks are [b_begin, b_end)
    if (b_begin >= need_max) {                   // no keys for this split: only keep the cluster barriers whole
        if (a.cluster_combine) { cluster_sync_all(); cluster_sync_all(); cluster_sync_all(); }
        return;
    }
    const int b_end = min(b_begin + a.split_units, need_max);
    const int nt_max = (b_end - b_begin + kTileBlks - 1) / kTileBlks;
#pragma unroll
    for (int m = 0; m < 2; ++m) nt[m] = max(0, (min(b_end, need[m]) - b_begin + kTileBlks - 1) / kTileBlks);
    const int ns_act = (need_max + a.split_units - 1) / a.split_units;        // CTAs of the pair that hold keys

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t bar_full = smem_u32(&bars->full[0]), bar_empty = smem_u32(&bars->empty[0]);
    const uint32_t bar_s = smem_u32(&bars->s_ready[0]), bar_p = smem_u32(&bars->p_ready[0]);
    const uint32_t bar_q = smem_u32(&bars->q_ready[0]), bar_scat = smem_u32(&bars->scat_done);
    const uint32_t bar_recv = smem_u32(&bars->recv);
    const uint32_t q_smem = base + P::kQOff, ring = base + P::kRingOff;

    // Producer warp, lanes 0-7: where block (tile's first block + lane) of this sequence lives.  The
    // block-table read of the FIRST tile is issued here, before the set-up barriers, so that its
    // latency (all CTAs of a launch hit the same table lines at once) is off the critical path.
    // With a.pdl this read (an __ldg) comes BEFORE griddepcontrol.wait, i.e. possibly while the previous
    // kernel of the stream still runs: swiftcache.h therefore requires the table to be complete before
    // that kernel starts.  Everything else the previous kernel may write is read after the wait.
    auto block_ptr = [&](int tb) -> const char * {
        const int lb = min(tb + lane, b_end - 1);
        // a resident block (regular cache) is read in place, the rest from the LSC
        return (a.has_res && lb < b.rc_blk[s])
                   ? a.kv_res.base + sc_phys_block(a.kv_res, b, s, lb) * a.kv_res.block_stride
                   : a.kv.base + sc_phys_block(a.kv, b, s, lb) * a.kv.block_stride;
    };
    const char *blk_next = (warp == 0 && lane < kTileBlks) ? block_ptr(b_begin) : nullptr;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kStages; ++i) { mbar_init(bar_full + 8 * i, 1); mbar_init(bar_empty + 8 * i, 1); }
        for (int m = 0; m < 2; ++m) {
            mbar_init(bar_s + 8 * m, 1);
            mbar_init(bar_p + 8 * m, kTM);
            mbar_init(bar_q + 8 * m, kTM);
            mbar_init(smem_u32(&bars->q_stage[m]), 1);
        }
        mbar_init(bar_scat, a.cluster_combine ? 64 * ns_act : 256);
        mbar_init(bar_recv, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 2) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;"
                     :: "r"(smem_u32(&bars->tmem_base)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    if (a.cluster_combine) cluster_sync_all();      // peers arrive on this CTA's barriers: they must exist
    else __syncthreads();
    tc_fence_after();
    const uint32_t tmem = bars->tmem_base;
    // Programmatic dependent launch: everything above overlapped the tail of the kernel before this
    // one in the stream; nothing below may start until that kernel's memory is visible (q, k_new,
    // v_new of this layer come from it in a model).  Then let the NEXT kernel begin its own set-up.
    // (Moving the wait to the top of the kernel, to start the Q loads earlier, was measured: it gives
    // up the overlap of the set-up with the previous kernel's tail, 1.18 -> 1.31 ms per fused turn.)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    float fin_m = -INFINITY, fin_l = 0.f;      // softmax threads: final (m in log2 units, l) of their row

    // ---- scatter (a5) ----
    // Every slot from T_h on of the blocks the pair reads is stored into the pool (and the LSC tail in
    // staged mode): the new tokens and, behind the sequence's last token, zeros, so that slots past the
    // logical end hold finite values whatever the memory held before (they are masked in S, but
    // 0 * NaN in P.V would poison the row).
    // Without a cluster (one CTA per pair): the softmax warps do it first, overlapped with the Q loads.
    // With a cluster (one CTA per split of this query pair and head): the rows are dealt out evenly
    // over the cluster's CTAs, whose otherwise idle warps 2-3 store them in the background, and each
    // thread then arrives (release, cluster scope) on the scat_done barrier of every CTA of the
    // cluster; a producer waits for all of them before it loads the first KV tile that holds new
    // tokens.  The host folds the scatter into this kernel only where that leaves ONE writer per row
    // (no grouped-query heads, one query pair per sequence: sc_ops.cu); the code below does not rely
    // on it.
    auto scatter_share = [&](auto nthreads_c, int tid, auto &&after_first_loads) {
        constexpr int NT = decltype(nthreads_c)::value;
        if (a.k_new == nullptr) { after_first_loads(); return; }
        bool mid_done = false;
        // every slot from T_h to the end of the last block this pair reads: the new tokens (up to 15 of
        // the next pair, which share that block, included) and, behind the sequence's last token, zeros
        const int ntok = n_s;
        const int nall = 16 * need_max - T_h;                        // rows of [K rows ; V rows] are 2 * nall
        int rest_lo = 0, rest_hi = 2 * nall;
        if (a.cluster_combine) {
            const int per = (2 * nall + ns_act - 1) / ns_act;
            rest_lo = split * per; rest_hi = min(2 * nall, rest_lo + per);
        }
        if (rest_lo < rest_hi) {
            constexpr int CPR = D / 8;                              // 16-byte units per head row
            const int hk = h / (g.Hq / g.Hkv);
            constexpr int RPI = NT / CPR;                           // rows the NT threads cover per step
            constexpr int U = NT == 64 ? 4 : 8;
            const int c = tid % CPR;
            for (int r0 = rest_lo + tid / CPR; r0 < rest_hi; r0 += RPI * U) {
                int4 val[U];
#pragma unroll
                for (int k = 0; k < U; ++k) {
                    const int rest = r0 + k * RPI;
                    val[k] = make_int4(0, 0, 0, 0);
                    if (rest < rest_hi) {
                        const int kv = rest >= nall, t = rest - kv * nall;
                        if (t < ntok) {
                            const int64_t row = (int64_t)b.cu_new[s] + t;
                            val[k] = __ldg(reinterpret_cast<const int4 *>(
                                (const char *)(kv ? a.v_new : a.k_new) + ((row * g.Hkv + hk) * D + c * 8) * 2));
                        }
                    }
                }
                if (!mid_done) { after_first_loads(); mid_done = true; }   // overlaps this round trip
#pragma unroll
                for (int k = 0; k < U; ++k) {
                    const int rest = r0 + k * RPI;
                    if (rest < rest_hi) {
                        const int kv = rest >= nall, t = rest - kv * nall;
                        const int tok = T_h + t, lb = tok >> 4, slot = tok & 15;
                        const int64_t in_cell = (int64_t)(kv * g.Hkv + hk) * P::kChunk + sc_chunk_off(slot, c * 8, NH);
                        *reinterpret_cast<int4 *>(a.scat0.base + sc_phys_block(a.scat0, b, s, lb) * a.scat0.block_stride + in_cell) = val[k];
                        if (a.has_scat1)
                            *reinterpret_cast<int4 *>(a.scat1.base + sc_phys_block(a.scat1, b, s, lb) * a.scat1.block_stride + in_cell) = val[k];
                    }
                }
            }
            asm volatile("fence.proxy.async.global;" ::: "memory");    // generic-proxy stores before bulk-copy reads
        }
        if (!mid_done) after_first_loads();
        if (a.cluster_combine) {
            for (int dst = 0; dst < ns_act; ++dst)
                asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" :: "r"(mapa(bar_scat, dst)) : "memory");
        } else {
            mbar_arrive(bar_scat);
        }
    };

    // registers: the producer / MMA warpgroup gives most of its share to the softmax warpgroups
    if (warp < 4) {
    if (LEAN) asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    else asm volatile("setmaxnreg.dec.sync.aligned.u32 72;");
    if (warp == 0) {
        // =============================== producer ===============================
        // Lane 0 owns the ring protocol (waits for a free slot, arms the full barrier); lanes 0-7 each
        // look up ONE block of the tile in the block table and issue its two bulk copies, and read
        // the table for the next tile while this one's copies are in flight.
        {
            const int hk = h / (g.Hq / g.Hkv);
            const int64_t off_kv[2] = {(int64_t)hk * P::kChunk, (int64_t)(g.Hkv + hk) * P::kChunk};
            bool scat_waited = (a.k_new == nullptr);
            // staged mode: an LSC line is read exactly once per layer -- after that it may go first
            uint64_t pol_stream = 0;
            if (LEAN) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol_stream));
            for (int jj = 0; jj < nt_max; ++jj) {
                const int tb = b_begin + jj * kTileBlks;         // first block of the tile
                const int nbt = min(kTileBlks, b_end - tb);      // blocks it holds
                const char *blk = blk_next;
                if (jj + 1 < nt_max && lane < kTileBlks) blk_next = block_ptr(tb + kTileBlks);
                if (!scat_waited && tb + nbt > (T_h >> 4)) {     // first tile with a block the scatter touches
                    if (lane == 0) mbar_wait_cluster(bar_scat, 0);
                    __syncwarp();
                    asm volatile("fence.proxy.async.global;" ::: "memory");   // generic-proxy stores -> bulk-copy reads
                    scat_waited = true;
                }
#pragma unroll
                for (int kv = 0; kv < 2; ++kv) {
                    const int it = 2 * jj + kv, slot = it % kStages;
                    if (lane == 0) {
                        mbar_wait(bar_empty + 8 * slot, ((it / kStages) & 1) ^ 1);
                        mbar_expect_tx(bar_full + 8 * slot, (uint32_t)nbt * P::kChunk);
                    }
                    __syncwarp();
                    if (lane < nbt) {
                        if (LEAN) bulk_g2s_hint(ring + slot * P::kSlot + lane * P::kChunk, blk + off_kv[kv], P::kChunk, bar_full + 8 * slot, pol_stream);
                        else bulk_g2s(ring + slot * P::kSlot + lane * P::kChunk, blk + off_kv[kv], P::kChunk, bar_full + 8 * slot);
                    }
                    if (it == 0 && lane == 0) {
                        // The first MMA needs Q and K of tile 0 only.  All CTAs start together, so
                        // the rest of the ring is requested once Q has landed: it would only queue
                        // in front of Q at the memory controllers.
#pragma unroll
                        for (int m = 0; m < 2; ++m)
                            if (nt[m] > 0) mbar_wait(bar_q + 8 * m, 0);
                    }
                }
            }
        }
        __syncwarp();
    } else if (warp == 1) {
        // =============================== MMA issuer ===============================
        if (lane == 0) {
            auto issue_qk = [&](int m, uint32_t kslot, int nbt) {
                const uint32_t idesc_qk = make_idesc(16 * nbt, 0);
#pragma unroll
                for (int hf = 0; hf < NH; ++hf)
#pragma unroll
                    for (int kk = 0; kk < 4; ++kk) {
                        const uint32_t o = hf * 1024 + kk * 32;
                        umma_ss(tmem + m * 128, make_desc(q_smem + m * P::kQTile + o, 16, NH * 1024),
                                make_desc(kslot + o, 16, NH * 1024), idesc_qk, (hf | kk) != 0);
                    }
            };
            auto issue_pv = [&](int m, uint32_t vslot, bool acc, int nbt) {
                constexpr uint32_t idesc_pv = make_idesc(D, 1);
#pragma unroll
                for (int kk = 0; kk < kTileBlks; ++kk)             // one MMA consumes one pool block
                    if (kk < nbt)
                        umma_ts(tmem + 256 + m * 128, tmem + m * 128 + kk * 8,
                                make_desc(vslot + kk * P::kChunk, 1024, NH * 1024), idesc_pv, acc || kk != 0);
            };
            auto slot_addr = [&](int it) { return ring + (it % kStages) * P::kSlot; };
            auto wait_full = [&](int it) {
                mbar_wait(bar_full + 8 * (it % kStages), (it / kStages) & 1);
                tc_fence_after();
            };
            auto blocks_of = [&](int jj) { return min(kTileBlks, b_end - (b_begin + jj * kTileBlks)); };
            // prologue: S_m = Q_m K_0^T
            wait_full(0);
#pragma unroll
            for (int m = 0; m < 2; ++m)
                if (nt[m] > 0) {
                    mbar_wait(bar_q + 8 * m, 0);
                    issue_qk(m, slot_addr(0), blocks_of(0));
                    umma_commit(bar_s + 8 * m);
                }
            umma_commit(bar_empty + 8 * (0 % kStages));
            for (int jj = 0; jj < nt_max; ++jj) {
                const int itv = 2 * jj + 1, itk = 2 * jj + 2;
                wait_full(itv);
                bool k_waited = false;
#pragma unroll
                for (int m = 0; m < 2; ++m) {
                    if (jj >= nt[m]) continue;
                    mbar_wait(bar_p + 8 * m, jj & 1);
                    tc_fence_after();
                    issue_pv(m, slot_addr(itv), jj > 0, blocks_of(jj));
                    if (jj + 1 < nt[m]) {
                        if (!k_waited) { wait_full(itk); k_waited = true; }
                        issue_qk(m, slot_addr(itk), blocks_of(jj + 1));
                    }
                    umma_commit(bar_s + 8 * m);      // S_m(jj+1) ready, or: O_m final
                }
                umma_commit(bar_empty + 8 * (itv % kStages));
                if (jj + 1 < nt_max) umma_commit(bar_empty + 8 * (itk % kStages));
            }
        }
        __syncwarp();
    } else if (a.cluster_combine) {
        // warps 2-3: this CTA's share of the cluster's scatter, in the background
        scatter_share(std::integral_constant<int, 64>{}, threadIdx.x - 64, []() {});
    }
    } else {
        // =============================== softmax warpgroups ===============================
        if (LEAN) asm volatile("setmaxnreg.inc.sync.aligned.u32 200;");
        else asm volatile("setmaxnreg.inc.sync.aligned.u32 208;");
        const int m = (warp - 4) >> 2, wl = warp & 3;
        const int r = wl * 32 + lane;                         // row of the query tile = TMEM lane
        const int t128 = threadIdx.x - 128 - m * kTM;         // 0..127 inside the warpgroup
        const int row0 = tok0 + m * kTM;                      // first new-token index of the tile
        const int64_t grow = (int64_t)b.cu_new[s] + row0 + r; // packed row of (s, token)
        {
            // ---- Q_m -> shared memory, swizzled exactly like a K tile.  The rows travel by the TMA engine
            //      (one 2*D-byte bulk copy per row, issued by the thread that owns the row) into ring slot
            //      1 + m, which the producer does not use before Q has landed; the warpgroup then moves them
            //      into place.  (Through the LSU path the 64 KB of Q took ~5k cycles: every SM starts
            //      streaming K/V at the same moment, and an SM's pending-request capacity over the loaded
            //      latency is ~11 B/clk.) ----
            constexpr int CPR = D / 8;                        // 16-byte units per row
            const uint32_t qs = q_smem + m * P::kQTile;
            const uint32_t stage = ring + (1 + m) * P::kSlot, bar_qs = smem_u32(&bars->q_stage[m]);
            if (nt[m] > 0) {
                if (t128 == 0) mbar_expect_tx(bar_qs, (uint32_t)rows[m] * (D * 2));
                if (r < rows[m])
                    bulk_g2s(stage + r * (D * 2), (const char *)a.q + (grow * g.Hq + h) * (D * 2), D * 2, bar_qs);
            }
            auto store_q = [&]() {
                if (nt[m] > 0) {
                    mbar_wait(bar_qs, 0);
#pragma unroll
                    for (int it = 0; it < CPR; ++it) {
                        const int u = it * kTM + t128;
                        const int row = u / CPR, c16 = u % CPR, hf = c16 >> 3, c = c16 & 7;
                        uint32_t v0 = 0, v1 = 0, v2 = 0, v3 = 0;
                        if (row < rows[m])
                            asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                                         : "=r"(v0), "=r"(v1), "=r"(v2), "=r"(v3) : "r"(stage + row * (D * 2) + c16 * 16));
                        const uint32_t dst = qs + (row >> 3) * (NH * 1024) + hf * 1024 + (row & 7) * 128 + ((c ^ (row & 7)) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};"
                                     :: "r"(dst), "r"(v0), "r"(v1), "r"(v2), "r"(v3) : "memory");
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // before the MMAs read Q and before V of tile 0 lands on the staging slot
                    mbar_arrive(bar_q + 8 * m);
                }
            };
            // without a cluster the softmax warps also do the scatter, overlapped with the Q loads
            if (a.cluster_combine) store_q();
            else scatter_share(std::integral_constant<int, 256>{}, threadIdx.x - 128, store_q);
        }

        const float sl = 1.4426950408889634f * rsqrtf((float)D);      // log2(e)/sqrt(D)
        const uint32_t lane_base = (uint32_t)(wl * 32) << 16;
        const uint32_t s_addr = tmem + lane_base + m * 128, o_addr = tmem + lane_base + 256 + m * 128;
        float m_used = -INFINITY, l_run = 0.f;
        for (int jj = 0; jj < nt[m]; ++jj) {
            const int tb = b_begin + jj * kTileBlks;
            const int ncols = 16 * min(kTileBlks, b_end - tb);   // keys in this tile
            mbar_wait(bar_s + 8 * m, jj & 1);
            tc_fence_after();
            // last visible column of this row inside the tile; columns past the tile's keys hold
            // stale values, so a tile with fewer than 128 keys is treated as masked
            const int limit = min(T_h + row0 + r - 16 * tb, ncols - 1);
            const bool masked_tile = (16 * tb + ncols - 1 > T_h + row0) || ncols < kTN;
            // S of this row: all columns at once (one tcgen05.wait::ld per tile), masked where the tile
            // crosses the causal boundary or holds fewer than 128 keys.
            uint32_t sv[kTN];
#pragma unroll
            for (int c4 = 0; c4 < kTN / 32; ++c4)
                tmem_ld32(s_addr + c4 * 32, *reinterpret_cast<uint32_t(*)[32]>(&sv[c4 * 32]));
            tmem_ld_wait();
            if (masked_tile) {
#pragma unroll
                for (int c = 0; c < kTN; ++c)
                    if (c > limit) sv[c] = 0xff800000u;             // -inf
            }
            float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};     // 4 chains: ILP
#pragma unroll
            for (int c = 0; c < kTN; c += 8)
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    mx4[k] = max3(mx4[k], __uint_as_float(sv[c + 2 * k]), __uint_as_float(sv[c + 2 * k + 1]));
            const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3]));
            const float m_new = fmaxf(m_used, mx);
            // P = 2^(s*sl - m_used*sl).  The reference m_used is LAZY: it is only advanced (and O
            // rescaled) when the row max has grown by more than 2^8, so P <= 256.
            const bool grow_max = (m_new - m_used) * sl > kRescaleThreshold;   // false for -inf - -inf (NaN)
            if (jj == 0) {
                m_used = m_new;                                     // O_m not accumulated yet
            } else if (__any_sync(0xffffffffu, grow_max)) {
                const float alpha = grow_max ? exp2f((m_used - m_new) * sl) : 1.f;
                if (grow_max) m_used = m_new;
                l_run *= alpha;
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait(o);
#pragma unroll
                    for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                    tmem_st32(o_addr + c4 * 32, o);
                }
            }
            const float msl = (m_used == -INFINITY) ? 0.f : m_used * sl;
            // two columns at a time (FFMA2 / FADD2)
            const uint64_t sl2 = pk2(sl, sl), nmsl2 = pk2(-msl, -msl);
            uint64_t rs2[2] = {0ull, 0ull};                         // (0.f, 0.f)
#pragma unroll
            for (int c = 0; c < kTN / 2; ++c) {
                uint64_t x = fma2(pk2(__uint_as_float(sv[2 * c]), __uint_as_float(sv[2 * c + 1])), sl2, nmsl2);
                float p0, p1;
                upk2(x, p0, p1);
                p0 = exp2f(p0);
                p1 = exp2f(p1);
                x = pk2(p0, p1);
                rs2[c & 1] = add2(rs2[c & 1], x);
                sv[c] = pack_bf16(p0, p1);                          // in place: c <= 2c
            }
            {
                float a0, a1, b0, b1;
                upk2(rs2[0], a0, a1);
                upk2(rs2[1], b0, b1);
                l_run += (a0 + a1) + (b0 + b1);
            }
            tmem_st32(s_addr, *reinterpret_cast<uint32_t(*)[32]>(&sv[0]));
            if (ncols > 64) tmem_st32(s_addr + 32, *reinterpret_cast<uint32_t(*)[32]>(&sv[32]));
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(bar_p + 8 * m);
        }

        fin_m = m_used * sl;
        fin_l = l_run;
        // ---- epilogue ----
        if (nt[m] > 0) {
            mbar_wait(bar_s + 8 * m, nt[m] & 1);
            tc_fence_after();
            const bool valid = r < rows[m];
            if (a.cluster_combine) {
                // O_m stays in TMEM until the cluster exchange below
            } else if (a.n_splits == 1) {
                const float inv = __fdividef(1.f, l_run);
                char *orow = (char *)a.out + (grow * g.Hq + h) * (D * 2);
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait(o);
                    if (valid) {
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4) {
                            int4 v;
                            v.x = pack_bf16(__uint_as_float(o[q4 * 8 + 0]) * inv, __uint_as_float(o[q4 * 8 + 1]) * inv);
                            v.y = pack_bf16(__uint_as_float(o[q4 * 8 + 2]) * inv, __uint_as_float(o[q4 * 8 + 3]) * inv);
                            v.z = pack_bf16(__uint_as_float(o[q4 * 8 + 4]) * inv, __uint_as_float(o[q4 * 8 + 5]) * inv);
                            v.w = pack_bf16(__uint_as_float(o[q4 * 8 + 6]) * inv, __uint_as_float(o[q4 * 8 + 7]) * inv);
                            *reinterpret_cast<int4 *>(orow + c4 * 64 + q4 * 16) = v;
                        }
                    }
                }
            } else {
                // The partial goes to the scratch buffer for sc_combine_kernel in the same form as in the
                // cluster exchange below: O scaled per row by a power of two 2^-e so that the largest element
                // lands in [8192, 16384), rounded to fp16, with (A, L) = (m + e, l * 2^-e) -- half the bytes of
                // fp32 partials for the kernel that writes them and for the one that reads them.
                const int64_t prow = ((int64_t)split * a.total_new + grow) * g.Hq + h;
                __half *orow = reinterpret_cast<__half *>(a.part_o) + prow * D;
                float amax = 0.f;
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait(o);
#pragma unroll
                    for (int c = 0; c < 32; c += 2)
                        amax = max3(amax, fabsf(__uint_as_float(o[c])), fabsf(__uint_as_float(o[c + 1])));
                }
                int e = (int)((__float_as_uint(amax) >> 23) & 0xffu) - 140;
                e = amax > 0.f ? max(e, -100) : 0;                              // all-zero rows keep e = 0
                const float scale = __uint_as_float((uint32_t)(127 - e) << 23); // 2^-e
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait(o);
                    if (valid) {
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4)
                            *reinterpret_cast<uint4 *>(orow + c4 * 32 + q4 * 8) = make_uint4(
                                pack_f16(__uint_as_float(o[q4 * 8 + 0]) * scale, __uint_as_float(o[q4 * 8 + 1]) * scale),
                                pack_f16(__uint_as_float(o[q4 * 8 + 2]) * scale, __uint_as_float(o[q4 * 8 + 3]) * scale),
                                pack_f16(__uint_as_float(o[q4 * 8 + 4]) * scale, __uint_as_float(o[q4 * 8 + 5]) * scale),
                                pack_f16(__uint_as_float(o[q4 * 8 + 6]) * scale, __uint_as_float(o[q4 * 8 + 7]) * scale));
                    }
                }
                if (valid) {
                    a.part_ml[prow * 2 + 0] = m_used * sl + (float)e;      // log2 units; may be -inf
                    a.part_ml[prow * 2 + 1] = l_run * scale;
                }
            }
        } else if (a.n_splits > 1 && !a.cluster_combine && r < rows[m]) {
            // the tile exists but sees none of this split's keys: weight 0 in the combine
            const int64_t prow = ((int64_t)split * a.total_new + grow) * g.Hq + h;
            a.part_ml[prow * 2 + 0] = -INFINITY;
            a.part_ml[prow * 2 + 1] = 0.f;
        }
    }

    // ---- split-KV combine (a7), in kernel.  The CTAs of one (query tile pair, head) form a
    //      thread-block cluster, one CTA per split, and each CTA is responsible for a slice of the
    //      pair's rows.  A CTA writes its partial into its own shared memory, one row per query row:
    //      O scaled by a power of two 2^-e chosen per row so that the largest element lands in
    //      [8192, 16384), rounded to fp16 (11 significant bits whatever the magnitude of V), and the
    //      pair (A, L) = (m + e, l * 2^-e), so that out = sum_s 2^A_s O16_s / sum_s 2^A_s L_s.  The
    //      TMA engine then copies each peer's slice into that peer's shared memory (one bulk copy per
    //      peer for O, one for (A, L), completing on the peer's mbarrier), and every CTA merges what it
    //      received in split order, so the result does not depend on timing. ----
    if (a.cluster_combine) {
        constexpr int CH = D / 8;                                  // 16-byte units per fp16 row
        const int nrows = min(kPairM, n_s - tok0);
        const int per = (((nrows + ns_act - 1) / ns_act) + 1) & ~1; // rows per CTA, even: (A, L) slices stay 16-byte units
        const int r_begin = min(nrows, split * per), n_mine = min(nrows, r_begin + per) - r_begin;
        const uint32_t stage_o = q_smem, stage_ml = base + P::kMlOff;
        const uint32_t recv_o = ring, recv_ml = ring + P::kRecvMlOff;
        if (threadIdx.x == 128)         // arm before any peer can send: everything the other CTAs owe this one
            mbar_expect_tx(bar_recv, (uint32_t)((ns_act - 1) * (n_mine * P::kRowB + ((n_mine + 1) & ~1) * 8)));
        cluster_arrive();               // this CTA's ring is free (softmax threads arrive after the last MMA)
        if (warp >= 4) {
            const int m = (warp - 4) >> 2, wl = warp & 3;
            const int prow = m * kTM + wl * 32 + lane;             // row of the pair
            const uint32_t o_addr = tmem + ((uint32_t)(wl * 32) << 16) + 256 + m * 128;
            const uint32_t dst_row = stage_o + (uint32_t)prow * P::kRowB;
            float stA = -INFINITY, stL = 0.f;                       // a tile that sees none of this split's keys: weight 0
            if (nt[m] > 0) {
                float amax = 0.f;
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait(o);
#pragma unroll
                    for (int c = 0; c < 32; c += 2)
                        amax = max3(amax, fabsf(__uint_as_float(o[c])), fabsf(__uint_as_float(o[c + 1])));
                }
                // 2^e = the power of two that brings amax into [8192, 16384); all-zero rows keep e = 0
                int e = (int)((__float_as_uint(amax) >> 23) & 0xffu) - 140;
                e = amax > 0.f ? max(e, -100) : 0;
                const float scale = __uint_as_float((uint32_t)(127 - e) << 23);       // 2^-e
                stA = fin_m + (float)e;
                stL = fin_l * scale;
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait(o);
#pragma unroll
                    for (int q = 0; q < 4; ++q) {                  // 8 values = one 16-byte unit
                        const uint32_t u = (uint32_t)((c4 * 4 + q) ^ (prow & (CH - 1)));
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};"
                                     :: "r"(dst_row + (u << 4)),
                                        "r"(pack_f16(__uint_as_float(o[q * 8 + 0]) * scale, __uint_as_float(o[q * 8 + 1]) * scale)),
                                        "r"(pack_f16(__uint_as_float(o[q * 8 + 2]) * scale, __uint_as_float(o[q * 8 + 3]) * scale)),
                                        "r"(pack_f16(__uint_as_float(o[q * 8 + 4]) * scale, __uint_as_float(o[q * 8 + 5]) * scale)),
                                        "r"(pack_f16(__uint_as_float(o[q * 8 + 6]) * scale, __uint_as_float(o[q * 8 + 7]) * scale))
                                     : "memory");
                    }
                }
            }
            asm volatile("bar.sync 1, 256;" ::: "memory");                 // both query tiles' MMAs are done: the ring is free
            asm volatile("st.shared.v2.f32 [%0], {%1, %2};" :: "r"(stage_ml + (uint32_t)prow * 8), "f"(stA), "f"(stL) : "memory");
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // these stores -> the TMA engine's reads
            asm volatile("bar.sync 1, 256;" ::: "memory");                 // the 8 softmax warps
        }
        cluster_wait();                 // every CTA of the cluster is done with its ring and has armed its barrier
        if (threadIdx.x == 128) {
            for (int d = 1; d < ns_act; ++d) {                     // start with the next CTA: spreads the traffic
                const int dst = (split + d) % ns_act;
                const int d_begin = min(nrows, dst * per), n_dst = min(nrows, d_begin + per) - d_begin;
                if (n_dst <= 0) continue;
                const uint32_t pbar = mapa(bar_recv, dst);
                bulk_s2peer(mapa(recv_o + (uint32_t)(split * per) * P::kRowB, dst), stage_o + (uint32_t)d_begin * P::kRowB,
                            (uint32_t)n_dst * P::kRowB, pbar);
                bulk_s2peer(mapa(recv_ml + (uint32_t)(split * per) * 8, dst), stage_ml + (uint32_t)d_begin * 8,
                            (uint32_t)((n_dst + 1) & ~1) * 8, pbar);
            }
        }
        if (warp >= 4) {
            mbar_wait_cluster(bar_recv, 0);
        }
        cluster_arrive();               // what this CTA had to receive has landed (so its senders' reads are done)
        if (warp >= 4 && n_mine > 0) {
            constexpr int RW = 32 / CH;                            // rows a warp handles per step
            const int w8 = warp - 4, u = lane % CH;
            for (int i = w8 * RW + lane / CH; i < n_mine; i += 8 * RW) {
                const int prow = r_begin + i;
                // split sp's partial of this row: own slice from the staging area, the others as received
                auto ml_addr = [&](int sp) {
                    return sp == split ? stage_ml + (uint32_t)prow * 8 : recv_ml + (uint32_t)(sp * per + i) * 8;
                };
                auto o_addr_of = [&](int sp) {
                    return (sp == split ? stage_o + (uint32_t)prow * P::kRowB : recv_o + (uint32_t)(sp * per + i) * P::kRowB) +
                           ((uint32_t)u << 4);
                };
                float Amax = -INFINITY;
                for (int sp = 0; sp < ns_act; ++sp) {
                    float A;
                    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(A) : "r"(ml_addr(sp)));
                    Amax = fmaxf(Amax, A);
                }
                float acc[8], W = 0.f;
#pragma unroll
                for (int k = 0; k < 8; ++k) acc[k] = 0.f;
                for (int sp0 = 0; sp0 < ns_act; sp0 += 4) {        // splits in order, four loads in flight
                    float A[4], L[4];
                    uint4 v[4];
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const int sp = min(sp0 + q, ns_act - 1);
                        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(A[q]), "=f"(L[q]) : "r"(ml_addr(sp)));
                        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                                     : "=r"(v[q].x), "=r"(v[q].y), "=r"(v[q].z), "=r"(v[q].w) : "r"(o_addr_of(sp)));
                        if (sp0 + q >= ns_act) A[q] = -INFINITY;
                    }
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        const bool on = A[q] != -INFINITY;         // a split that sent no O leaves stale but unused bytes
                        const float wgt = on ? exp2f(A[q] - Amax) : 0.f;
                        W += on ? wgt * L[q] : 0.f;
                        const uint32_t w4[4] = {v[q].x, v[q].y, v[q].z, v[q].w};
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const float2 f = unpack_f16(w4[k]);
                            acc[2 * k] += on ? wgt * f.x : 0.f;
                            acc[2 * k + 1] += on ? wgt * f.y : 0.f;
                        }
                    }
                }
                const float inv = __fdividef(1.f, W);
                uint4 o4;
                o4.x = pack_bf16(acc[0] * inv, acc[1] * inv);
                o4.y = pack_bf16(acc[2] * inv, acc[3] * inv);
                o4.z = pack_bf16(acc[4] * inv, acc[5] * inv);
                o4.w = pack_bf16(acc[6] * inv, acc[7] * inv);
                const int64_t grow = (int64_t)b.cu_new[s] + tok0 + prow;
                const int c = u ^ (prow & (CH - 1));               // un-swizzle: which 8 columns this unit holds
                *reinterpret_cast<uint4 *>((char *)a.out + (grow * g.Hq + h) * (D * 2) + c * 16) = o4;
            }
        }
        cluster_wait();                 // no CTA leaves while a peer's copy may still read its shared memory
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tmem) : "memory");
}

}  // namespace

int sc_tc_tile_m() { return kPairM; }
int sc_tc_split_unit() { return 16; }          // splits are in pool blocks

template <int D, int LEAN>
static cudaError_t prepare_tc()
{
    static std::atomic<uint64_t> done{0};
    if (!sc_first_use_on_device(done)) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(sc_attn_tc_kernel<D, LEAN>, cudaFuncAttributeMaxDynamicSharedMemorySize, Plan<D>::kBytes);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(sc_attn_tc_kernel<D, LEAN>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    return e;
}

template <int D, int LEAN>
static void fill_config(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr, dim3 grid, int cluster, bool pdl, cudaStream_t st)
{
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = grid;
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = Plan<D>::kBytes;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = cluster;                               // one CTA per split
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    // Programmatic dependent launch: this kernel may be scheduled while the kernel before it in the
    // stream drains; it waits (griddepcontrol.wait) before it touches anything that kernel wrote.
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 2 : 1;
}

template <int D, int LEAN>
static cudaError_t launch_tc(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, dim3 grid, cudaStream_t st)
{
    cudaError_t e = prepare_tc<D, LEAN>();
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[2];
    fill_config<D, LEAN>(cfg, attr, grid, a.cluster_combine ? (int)grid.x : 1, a.pdl != 0, st);
    return cudaLaunchKernelEx(&cfg, sc_attn_tc_kernel<D, LEAN>, g, b, a);
}

// CTAs that can be resident at once when the kernel is launched in clusters of `cluster` CTAs
// (each CTA needs a whole SM; a cluster must fit in one GPC).  0 if such clusters cannot launch.
template <int D, int LEAN>
static int wave_ctas(int cluster)
{
    if (prepare_tc<D, LEAN>() != cudaSuccess) return 0;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[2];
    fill_config<D, LEAN>(cfg, attr, dim3((unsigned)cluster, 1, 1), cluster, false, nullptr);
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, sc_attn_tc_kernel<D, LEAN>, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return n * cluster;
}

int sc_tc_max_cluster() { return kMaxCluster; }

int sc_tc_wave_ctas(int D, int lean, int cluster)
{
    static int cache[SC_MAX_DEVICES][2][2][kMaxCluster + 1];          // 0 = not asked yet, -1 = cannot launch
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= SC_MAX_DEVICES) dev = 0;
    int &c = cache[dev][D == 128][lean != 0][cluster];
    if (c == 0) {
        const int n = D == 128 ? (lean ? wave_ctas<128, 1>(cluster) : wave_ctas<128, 0>(cluster))
                               : (lean ? wave_ctas<64, 1>(cluster) : wave_ctas<64, 0>(cluster));
        c = n > 0 ? n : -1;
    }
    return c > 0 ? c : 0;
}
cudaError_t sc_launch_attn_tc(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, cudaStream_t st)
{
    const int total_pairs = b.cu_mt[b.n_seq];
    if (total_pairs == 0) return cudaSuccess;
    dim3 grid((unsigned)a.n_splits, (unsigned)g.Hq, (unsigned)total_pairs);
    if (a.has_scat1)   // staged mode: a gather runs beside this kernel
        return g.D == 128 ? launch_tc<128, 1>(g, b, a, grid, st) : launch_tc<64, 1>(g, b, a, grid, st);
    return g.D == 128 ? launch_tc<128, 0>(g, b, a, grid, st) : launch_tc<64, 0>(g, b, a, grid, st);
}
