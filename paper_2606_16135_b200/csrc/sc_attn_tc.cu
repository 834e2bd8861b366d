// sc_attn_tc.cu -- paged prefill attention, tcgen05 / TMEM engine (
// each new token attends to all history tokens and to the new tokens up to
// and including itself).
//
// One CTA owns a PAIR of 128-row query tiles of one query head (256 new tokens) and a
// contiguous range of 128-token KV tiles (one split).  Warp roles:
//   warp 0      producer : per KV tile, 8 + 8 bulk copies (cp.async.bulk, 4 KiB each) bring
//                          the K and V chunks of the tile's 8 pool blocks -- found through the
//                          block table -- into a 5-slot shared-memory ring.  The pool stores
//                          chunks in the tensor core's 128B-swizzled operand order
//                          (include/swiftcache.h), so a chunk is an MMA operand as it lands.
//   warp 1      MMA      : one thread issues tcgen05.mma.  S_m = Q_m K^T (both operands in
//                          shared memory, K-major) into TMEM; O_m += P_m V with P_m read from
//                          TMEM and V as an MN-major shared-memory operand.
//   warp 2      TMEM allocation (all 512 columns: S0 S1 O0 O1, 128 fp32 columns each);
//   warps 2-3   in cluster mode: this CTA's share of the scatter of the new K/V (a5)
//   warps 4-7   softmax warpgroup of query tile 0: thread r owns row r.  tcgen05.ld S,
//   warps 8-11  same for query tile 1            : mask, online softmax in registers with
//                          lazy rescaling of O (only when the row max grows by > 2^8), P
//                          rounded to bf16 and stored over S in TMEM, epilogue.
// The two query tiles ping-pong on the tensor pipe: while warpgroup 0 does the softmax of
// tile j, the pipe runs PV and QK^T of query tile 1.
//
// Split-KV (a7): with up to 16 splits that fit one wave, the CTAs of one (query pair, head) are
// a thread-block cluster; they share the scatter and merge their partial (m, l, O) through
// distributed shared memory at the end.  Otherwise partials go to global scratch and
// sc_combine_kernel merges them, and the scatter kernel runs before this one.
//
// Work partitioning depends on logical positions only, so results are bit-identical under
// any permutation of physical block ids, and staged attention is this same kernel run with
// the identity table over the LSC.
#include <cuda_bf16.h>
#include <stdlib.h>

#include <type_traits>

#include "sc_internal.h"

namespace {

constexpr int kTM = 128;          // rows of one query tile
constexpr int kPairM = 2 * kTM;   // rows a CTA owns
constexpr int kTN = 128;          // KV tokens per tile (8 pool blocks)
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
// SC_ERR_CUDA on the next call) instead of spinning forever on a protocol error.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    long long t0 = 0;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        const long long t = clock64();
        if (t0 == 0) t0 = t;
        else if (t - t0 > 4000000000ll) __trap();
    }
}
// same, acquiring at cluster scope (the arrivals come from other CTAs of the cluster)
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    long long t0 = 0;
    for (;;) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
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

// all threads of all CTAs of the cluster; release / acquire at cluster scope (global writes included)
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

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

// shared-memory plan (offsets from the 1024-byte aligned base)
template <int D>
struct Plan {
    static constexpr int NH = D / 64;
    static constexpr int kChunk = 16 * D * 2;          // one (block, head) chunk
    static constexpr int kQTile = kTM * D * 2;         // one query tile, swizzled like a K tile
    static constexpr int kSlot = kTN * D * 2;          // K (or V) of one KV tile = 8 chunks
    static constexpr int kQOff = 0;
    static constexpr int kRingOff = 2 * kQTile;
    static constexpr int kBarOff = kRingOff + kStages * kSlot;
    static constexpr int kBytes = kBarOff + 256 + 1024;   // + barriers + alignment slack
};

struct Bars {                       // at Plan::kBarOff
    uint64_t full[kStages], empty[kStages];
    uint64_t s_ready[2];            // MMA -> softmax warpgroup m: S_m written (and earlier PV_m done)
    uint64_t p_ready[2];            // softmax warpgroup m -> MMA: P_m stored, O_m rescaled
    uint64_t q_ready[2];            // Q_m in shared memory
    uint64_t scat_done;             // warps 2-3 -> producer: this CTA's share of the new K/V is in the pool
    uint32_t tmem_base;
};

#ifdef SC_TC_PROBE
__constant__ int sc_probe_flags;
__device__ long long sc_tl[256][64];
#define PROBE(bit) (sc_probe_flags & (1 << (bit)))
#define TL(i) do { const int cta_ = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z); \
                   if (cta_ < 256) sc_tl[cta_][(i)] = clock64(); } while (0)
#define TLG(i) do { const int cta_ = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z); \
                    long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); \
                    if (cta_ < 256) sc_tl[cta_][(i)] = t_; } while (0)
#else
#define PROBE(bit) 0
#define TL(i) do { } while (0)
#define TLG(i) do { } while (0)
#endif

template <int D, int LEAN>
__global__ void __maxnreg__(LEAN ? 152 : 168)
sc_attn_tc_kernel(ScGeom g, ScBatch b, ScAttnArgs a)
{
    using P = Plan<D>;
    constexpr int NH = P::NH;
    extern __shared__ char smem_raw[];
    const uint32_t raw_u32 = smem_u32(smem_raw);
    const uint32_t base = (raw_u32 + 1023u) & ~1023u;
    char *smem = smem_raw + (base - raw_u32);
    Bars *bars = reinterpret_cast<Bars *>(smem + P::kBarOff);

    // ---- which work is this CTA's (all of it warp- and CTA-uniform) ----
    const int split = blockIdx.x, h = blockIdx.y, gp = blockIdx.z;
    const int s = seq_of(b.cu_mt, b.n_seq, gp);
    const int pair = gp - b.cu_mt[s];
    const int n_s = b.cu_new[s + 1] - b.cu_new[s];
    const int T_h = b.hist[s];
    const int tok0 = pair * kPairM;
    int rows[2], need[2], nt[2];
#pragma unroll
    for (int m = 0; m < 2; ++m) {
        rows[m] = max(0, min(kTM, n_s - tok0 - m * kTM));
        need[m] = rows[m] > 0 ? (T_h + tok0 + m * kTM + rows[m] + kTN - 1) / kTN : 0;
    }
    const int need_max = max(need[0], need[1]);
    const int t_begin = split * a.split_tiles;
    if (t_begin >= need_max) {                   // no keys for this split: only keep the cluster barriers whole
        if (a.cluster_combine) { cluster_sync_all(); cluster_sync_all(); cluster_sync_all(); }
        return;
    }
    const int t_end = min(t_begin + a.split_tiles, need_max);
    const int nt_max = t_end - t_begin;
#pragma unroll
    for (int m = 0; m < 2; ++m) nt[m] = max(0, min(t_end, need[m]) - t_begin);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) { TL(0); TLG(60); }
    const uint32_t bar_full = smem_u32(&bars->full[0]), bar_empty = smem_u32(&bars->empty[0]);
    const uint32_t bar_s = smem_u32(&bars->s_ready[0]), bar_p = smem_u32(&bars->p_ready[0]);
    const uint32_t bar_q = smem_u32(&bars->q_ready[0]), bar_scat = smem_u32(&bars->scat_done);
    const uint32_t q_smem = base + P::kQOff, ring = base + P::kRingOff;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kStages; ++i) { mbar_init(bar_full + 8 * i, 1); mbar_init(bar_empty + 8 * i, 1); }
        for (int m = 0; m < 2; ++m) {
            mbar_init(bar_s + 8 * m, 1);
            mbar_init(bar_p + 8 * m, kTM);
            mbar_init(bar_q + 8 * m, kTM);
        }
        mbar_init(bar_scat, a.cluster_combine ? 64 * ((need_max + a.split_tiles - 1) / a.split_tiles) : 256);
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
    if (threadIdx.x == 128) TL(1);
    float fin_m = -INFINITY, fin_l = 0.f;      // softmax threads: final (m in log2 units, l) of their row

    // ---- scatter (a5) ----
    // Without a cluster: the softmax warps do it first; the CTA stores the new tokens at positions [p_lo, p_hi) -- those inside
    // its own KV tiles that its query tiles can see -- and only relies on its own stores.
    // With a cluster (one CTA per split of this query pair and head): the pair's new tokens are
    // dealt out evenly over the cluster's CTAs, whose otherwise idle warps 2-3 store them in the
    // background, and each thread then arrives (release, cluster
    // scope) on the scat_done barrier of every CTA of the cluster; a producer waits for all of
    // them before it loads the first KV tile that holds new tokens.  CTAs of other query heads
    // of the group or of later query pairs may store the same bytes to the same places.
    const int ns_act = (need_max + a.split_tiles - 1) / a.split_tiles;        // CTAs of the pair that hold keys
    auto scatter_share = [&](auto nthreads_c, int tid, auto &&after_first_loads) {
        constexpr int NT = decltype(nthreads_c)::value;
        if (a.k_new == nullptr) { after_first_loads(); return; }
        bool mid_done = false;
        const int ntok_pair = min(n_s, tok0 + kPairM);
        int p_lo, ntok, rest_lo, rest_hi;                            // rows of [K rows ; V rows] to store
        if (a.cluster_combine) {
            p_lo = T_h; ntok = ntok_pair;
            const int per = (2 * ntok + ns_act - 1) / ns_act;
            rest_lo = split * per; rest_hi = min(2 * ntok, rest_lo + per);
        } else {
            p_lo = max(T_h, kTN * t_begin); ntok = min(T_h + ntok_pair, kTN * t_end) - p_lo;
            rest_lo = 0; rest_hi = 2 * ntok;
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
                    if (rest < rest_hi) {
                        const int kv = rest >= ntok, t = rest - kv * ntok;
                        const int64_t row = (int64_t)b.cu_new[s] + (p_lo + t - T_h);
                        val[k] = __ldg(reinterpret_cast<const int4 *>(
                            (const char *)(kv ? a.v_new : a.k_new) + ((row * g.Hkv + hk) * D + c * 8) * 2));
                    }
                }
                if (!mid_done) { after_first_loads(); mid_done = true; }   // overlaps this round trip
#pragma unroll
                for (int k = 0; k < U; ++k) {
                    const int rest = r0 + k * RPI;
                    if (rest < rest_hi) {
                        const int kv = rest >= ntok, t = rest - kv * ntok;
                        const int tok = p_lo + t, lb = tok >> 4, slot = tok & 15;
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
            for (int dst = 0; dst < ns_act; ++dst) {
                uint32_t rbar;
                asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rbar) : "r"(bar_scat), "r"(dst));
                asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" :: "r"(rbar) : "memory");
            }
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
        if (lane == 0) {
            const int nblk = (T_h + n_s + 15) >> 4;
            const int hk = h / (g.Hq / g.Hkv);
            const int64_t off_kv[2] = {(int64_t)hk * P::kChunk, (int64_t)(g.Hkv + hk) * P::kChunk};
            bool scat_waited = (a.k_new == nullptr);
            for (int jj = 0; jj < nt_max; ++jj) {
                const int j = t_begin + jj;
                if (!scat_waited && j >= T_h / kTN) {      // first tile with a block the scatter touches
                    mbar_wait_cluster(bar_scat, 0);
                    asm volatile("fence.proxy.async.global;" ::: "memory");   // generic-proxy stores -> bulk-copy reads
                    scat_waited = true;
                }
                const char *blk[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    const int lb = min(j * 8 + c, nblk - 1);
                    // a resident block (regular cache) is read in place, the rest from the LSC
                    blk[c] = (a.has_res && lb < b.rc_blk[s])
                                 ? a.kv_res.base + sc_phys_block(a.kv_res, b, s, lb) * a.kv_res.block_stride
                                 : a.kv.base + sc_phys_block(a.kv, b, s, lb) * a.kv.block_stride;
                }
#pragma unroll
                for (int kv = 0; kv < 2; ++kv) {
                    const int it = 2 * jj + kv, slot = it % kStages;
                    mbar_wait(bar_empty + 8 * slot, ((it / kStages) & 1) ^ 1);
                    if (PROBE(4)) { mbar_arrive(bar_full + 8 * slot); continue; }
                    mbar_expect_tx(bar_full + 8 * slot, P::kSlot);
#pragma unroll
                    for (int c = 0; c < 8; ++c)
                        bulk_g2s(ring + slot * P::kSlot + c * P::kChunk, blk[c] + off_kv[kv], P::kChunk,
                                 bar_full + 8 * slot);
                    if (it == 0) {
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
            constexpr uint32_t idesc_qk = make_idesc(kTN, 0), idesc_pv = make_idesc(D, 1);
            auto issue_qk = [&](int m, uint32_t kslot) {
                if (PROBE(3)) return;
#pragma unroll
                for (int hf = 0; hf < NH; ++hf)
#pragma unroll
                    for (int kk = 0; kk < 4; ++kk) {
                        const uint32_t o = hf * 1024 + kk * 32;
                        umma_ss(tmem + m * 128, make_desc(q_smem + m * P::kQTile + o, 16, NH * 1024),
                                make_desc(kslot + o, 16, NH * 1024), idesc_qk, (hf | kk) != 0);
                    }
            };
            auto issue_pv = [&](int m, uint32_t vslot, bool acc) {
                if (PROBE(2)) return;
#pragma unroll
                for (int kk = 0; kk < 8; ++kk)
                    umma_ts(tmem + 256 + m * 128, tmem + m * 128 + kk * 8,
                            make_desc(vslot + kk * P::kChunk, 1024, NH * 1024), idesc_pv, acc || kk != 0);
            };
            auto slot_addr = [&](int it) { return ring + (it % kStages) * P::kSlot; };
            auto wait_full = [&](int it) {
                mbar_wait(bar_full + 8 * (it % kStages), (it / kStages) & 1);
                tc_fence_after();
            };
            // prologue: S_m = Q_m K_0^T
            wait_full(0);
#pragma unroll
            for (int m = 0; m < 2; ++m)
                if (nt[m] > 0) {
                    mbar_wait(bar_q + 8 * m, 0);
                    issue_qk(m, slot_addr(0));
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
                    issue_pv(m, slot_addr(itv), jj > 0);
                    if (jj + 1 < nt[m]) {
                        if (!k_waited) { wait_full(itk); k_waited = true; }
                        issue_qk(m, slot_addr(itk));
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
            // ---- Q_m -> shared memory, swizzled exactly like a K tile; its global loads and the
            //      first round of scatter loads share one memory round trip ----
            constexpr int CPR = D / 8;                        // 16-byte units per row
            const char *qg = (const char *)a.q;
            const uint32_t qs = q_smem + m * P::kQTile;
            int4 qv[CPR];
            if (nt[m] > 0) {
#pragma unroll
                for (int it = 0; it < CPR; ++it) {
                    const int u = it * kTM + t128;
                    const int row = u / CPR, c16 = u % CPR;
                    qv[it] = make_int4(0, 0, 0, 0);
                    if (row < rows[m])
                        qv[it] = __ldg(reinterpret_cast<const int4 *>(
                            qg + (((int64_t)b.cu_new[s] + row0 + row) * g.Hq + h) * (D * 2) + c16 * 16));
                }
            }
            auto store_q = [&]() {
                if (nt[m] > 0) {
#pragma unroll
                    for (int it = 0; it < CPR; ++it) {
                        const int u = it * kTM + t128;
                        const int row = u / CPR, c16 = u % CPR, hf = c16 >> 3, c = c16 & 7;
                        const uint32_t dst = qs + (row >> 3) * (NH * 1024) + hf * 1024 + (row & 7) * 128 + ((c ^ (row & 7)) << 4);
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};"
                                     :: "r"(dst), "r"(qv[it].x), "r"(qv[it].y), "r"(qv[it].z), "r"(qv[it].w) : "memory");
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                    mbar_arrive(bar_q + 8 * m);
                    if (threadIdx.x == 128) TL(2);
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
            const int j = t_begin + jj;
            mbar_wait(bar_s + 8 * m, jj & 1);
            tc_fence_after();
            if (threadIdx.x == 128 && jj < 12) TL(3 + 2 * jj);
            if (threadIdx.x == 256 && jj < 12) TL(40 + jj);
            if (PROBE(1)) { tc_fence_before(); mbar_arrive(bar_p + 8 * m); continue; }
            uint32_t sv[kTN];
#pragma unroll
            for (int c4 = 0; c4 < kTN / 32; ++c4)
                tmem_ld32(s_addr + c4 * 32, *reinterpret_cast<uint32_t(*)[32]>(&sv[c4 * 32]));
            tmem_ld_wait();
            if (j * kTN + kTN - 1 > T_h + row0) {               // tile reaches past the first row's limit
                const int limit = T_h + row0 + r - j * kTN;     // last visible column of this row
#pragma unroll
                for (int c = 0; c < kTN; ++c)
                    if (c > limit) sv[c] = 0xff800000u;         // -inf
            }
            if (PROBE(0)) {
                tmem_st32(s_addr, *reinterpret_cast<uint32_t(*)[32]>(&sv[0]));
                tmem_st32(s_addr + 32, *reinterpret_cast<uint32_t(*)[32]>(&sv[32]));
                tmem_st_wait();
                tc_fence_before();
                mbar_arrive(bar_p + 8 * m);
                continue;
            }
            float mx4[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};     // 4 chains: ILP
#pragma unroll
            for (int c = 0; c < kTN; c += 8)
#pragma unroll
                for (int k = 0; k < 4; ++k)
                    mx4[k] = fmaxf(mx4[k], fmaxf(__uint_as_float(sv[c + 2 * k]), __uint_as_float(sv[c + 2 * k + 1])));
            const float mx = fmaxf(fmaxf(mx4[0], mx4[1]), fmaxf(mx4[2], mx4[3]));
            const float m_new = fmaxf(m_used, mx);
            const bool grow_max = (m_new - m_used) * sl > kRescaleThreshold;   // false for -inf - -inf (NaN)
            if (jj == 0) {
                m_used = m_new;                                 // O_m not accumulated yet
            } else if (__any_sync(0xffffffffu, grow_max)) {
                const float alpha = grow_max ? exp2f((m_used - m_new) * sl) : 1.f;
                if (grow_max) m_used = m_new;
                l_run *= alpha;
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait();
#pragma unroll
                    for (int c = 0; c < 32; ++c) o[c] = __float_as_uint(__uint_as_float(o[c]) * alpha);
                    tmem_st32(o_addr + c4 * 32, o);
                }
            }
            const float msl = (m_used == -INFINITY) ? 0.f : m_used * sl;
            // P = 2^(s*sl - m*sl), two columns at a time.  (Moving a share of the exp2 to the FMA pipe
            // with a polynomial was measured slower at every share: with one softmax warp per
            // scheduler and query tile the loop is issue-bound, not MUFU-bound.)
            const uint64_t sl2 = pk2(sl, sl), nmsl2 = pk2(-msl, -msl);
            uint64_t rs2[2] = {0ull, 0ull};                     // (0.f, 0.f)
#pragma unroll
            for (int c = 0; c < kTN / 2; ++c) {
                uint64_t x = fma2(pk2(__uint_as_float(sv[2 * c]), __uint_as_float(sv[2 * c + 1])), sl2, nmsl2);
                float p0, p1;
                upk2(x, p0, p1);
                p0 = exp2f(p0);
                p1 = exp2f(p1);
                x = pk2(p0, p1);
                rs2[c & 1] = add2(rs2[c & 1], x);
                sv[c] = pack_bf16(p0, p1);                      // in place: c <= 2c
            }
            {
                float a0, a1, b0, b1;
                upk2(rs2[0], a0, a1);
                upk2(rs2[1], b0, b1);
                l_run += (a0 + a1) + (b0 + b1);
            }
            tmem_st32(s_addr, *reinterpret_cast<uint32_t(*)[32]>(&sv[0]));
            tmem_st32(s_addr + 32, *reinterpret_cast<uint32_t(*)[32]>(&sv[32]));
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(bar_p + 8 * m);
            if (threadIdx.x == 128 && jj < 12) TL(4 + 2 * jj);
        }

        fin_m = m_used * sl;
        fin_l = l_run;
        // ---- epilogue ----
        if (nt[m] > 0) {
            mbar_wait(bar_s + 8 * m, nt[m] & 1);
            tc_fence_after();
            if (threadIdx.x == 128) TL(30);
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
                    tmem_ld_wait();
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
                const int64_t prow = ((int64_t)split * a.total_new + grow) * g.Hq + h;
                float *orow = a.part_o + prow * D;
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait();
                    if (valid) {
#pragma unroll
                        for (int q4 = 0; q4 < 8; ++q4)
                            *reinterpret_cast<uint4 *>(orow + c4 * 32 + q4 * 4) =
                                make_uint4(o[q4 * 4], o[q4 * 4 + 1], o[q4 * 4 + 2], o[q4 * 4 + 3]);
                    }
                }
                if (valid) {
                    a.part_ml[prow * 2 + 0] = m_used * sl;      // log2 units; may be -inf
                    a.part_ml[prow * 2 + 1] = l_run;
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
    //      thread-block cluster, one CTA per split.  Each CTA is responsible for a slice of the
    //      pair's rows: every CTA sends the other CTAs' slices of its unnormalised partial
    //      (m, l, O) straight from TMEM into their shared memory (DSMEM), and merges what it
    //      receives in split order, so the result does not depend on timing. ----
    if (a.cluster_combine) {
        constexpr int CH = D / 4;                                  // 16-byte chunks per fp32 row
        const int ns = (need_max + a.split_tiles - 1) / a.split_tiles;     // CTAs that hold keys
        const int nrows = min(kPairM, n_s - tok0);
        const int per = (nrows + ns - 1) / ns;                     // rows per CTA
        const uint32_t recv_o = ring, recv_ml = ring + (kPairM + 16) * D * 4;   // [src][per][D] fp32, [src][per] (m, l)
        cluster_sync_all();                  // every CTA of the cluster is done with its ring
        if (threadIdx.x == 128) TL(31);
        if (warp >= 4) {
            const int m = (warp - 4) >> 2, wl = warp & 3;
            const int prow = m * kTM + wl * 32 + lane;             // row of the pair
            const bool valid = prow < nrows;
            const int dst = valid ? prow / per : 0, i = prow - dst * per;
            const uint32_t slot = (uint32_t)(split * per + i);
            uint32_t rem_o, rem_ml;
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rem_o) : "r"(recv_o + slot * (D * 4)), "r"(dst));
            asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rem_ml) : "r"(recv_ml + slot * 8), "r"(dst));
            if (valid)
                asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" :: "r"(rem_ml), "f"(nt[m] > 0 ? fin_m : -INFINITY),
                             "f"(nt[m] > 0 ? fin_l : 0.f) : "memory");
            if (nt[m] > 0) {
                // O rows go out through a per-warp 32 x 128-byte transposing scratch (in the idle Q
                // area), so that a remote store instruction writes four 128-byte runs instead of
                // 32 isolated 16-byte pieces.  Within a 128-byte run the 16-byte chunks are XORed
                // with (row & 7) -- conflict-free for the row-per-thread writes, and the same
                // order in the scratch and at the destination, so the read-out is a linear copy.
                const uint32_t o_addr = tmem + ((uint32_t)(wl * 32) << 16) + 256 + m * 128;
                const uint32_t scratch = q_smem + (uint32_t)(warp - 4) * 4096;
                uint32_t rem_row[8];                               // destination row of (it*4 + lane/8)
                bool ok_row[8];
#pragma unroll
                for (int it = 0; it < 8; ++it) {
                    const int pr = m * kTM + wl * 32 + it * 4 + (lane >> 3);
                    ok_row[it] = pr < nrows;
                    const int d = ok_row[it] ? pr / per : 0, ii = pr - d * per;
                    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(rem_row[it])
                                 : "r"(recv_o + (uint32_t)(split * per + ii) * (D * 4) + (lane & 7) * 16), "r"(d));
                }
#pragma unroll
                for (int c4 = 0; c4 < D / 32; ++c4) {
                    uint32_t o[32];
                    tmem_ld32(o_addr + c4 * 32, o);
                    tmem_ld_wait();
                    __syncwarp();                                  // previous read-out of the scratch is done
#pragma unroll
                    for (int q = 0; q < 8; ++q)
                        asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};"
                                     :: "r"(scratch + lane * 128 + (((uint32_t)q ^ (lane & 7)) << 4)), "r"(o[q * 4]), "r"(o[q * 4 + 1]),
                                        "r"(o[q * 4 + 2]), "r"(o[q * 4 + 3]) : "memory");
                    __syncwarp();
#pragma unroll
                    for (int it = 0; it < 8; ++it) {
                        uint32_t x, y, z, w;
                        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(x), "=r"(y), "=r"(z), "=r"(w)
                                     : "r"(scratch + it * 512 + lane * 16));
                        if (ok_row[it])
                            asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};"
                                         :: "r"(rem_row[it] + c4 * 128), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
                    }
                }
            }
        }
        if (threadIdx.x == 128) TL(32);
        cluster_sync_all();                  // all partials have landed
        if (threadIdx.x == 128) TL(34);
        if (warp >= 4) {
            constexpr int RW = 32 / CH;                            // rows a warp handles per step
            constexpr int RB = 4;                                  // steps in flight
            const int w8 = warp - 4, pch = lane % CH;
            const int r_begin = split * per, n_mine = min(nrows, r_begin + per) - r_begin;
            for (int i0 = w8 * RW + lane / CH; i0 < n_mine; i0 += 8 * RW * RB) {
                float Mrow[RB];
                // all loads first (unconditional: a split that sent no O leaves stale but unused bytes)
                float2 ml[RB][4];
                float4 v[RB][4];
                float4 acc[RB];
                float W[RB];
#pragma unroll
                for (int k = 0; k < RB; ++k) { acc[k] = make_float4(0.f, 0.f, 0.f, 0.f); W[k] = 0.f; }
#pragma unroll
                for (int sp0 = 0; sp0 < kMaxCluster; sp0 += 4) { // splits in order, four at a time
                    if (sp0 >= ns) break;
#pragma unroll
                    for (int k = 0; k < RB; ++k) {
                        const int i = min(i0 + k * 8 * RW, n_mine - 1);   // clamped duplicates are not written
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const int sp = min(sp0 + q, ns - 1);
                            asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(ml[k][q].x), "=f"(ml[k][q].y)
                                         : "r"(recv_ml + (uint32_t)(sp * per + i) * 8));
                            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];"
                                         : "=f"(v[k][q].x), "=f"(v[k][q].y), "=f"(v[k][q].z), "=f"(v[k][q].w)
                                         : "r"(recv_o + (uint32_t)(sp * per + i) * (D * 4) + pch * 16));
                            if (sp0 + q >= ns) ml[k][q] = make_float2(-INFINITY, 0.f);
                        }
                    }
                    // merge this group into the running (M, W, acc) of each row: the running max
                    // is the first group's max unless a later group raises it (rescale, rare)
#pragma unroll
                    for (int k = 0; k < RB; ++k) {
                        float Mg = fmaxf(fmaxf(ml[k][0].x, ml[k][1].x), fmaxf(ml[k][2].x, ml[k][3].x));
                        if (sp0 == 0) Mrow[k] = Mg;
                        else if (Mg > Mrow[k]) {
                            const float sc = exp2f(Mrow[k] - Mg);   // Mrow finite or -inf (then sc = 0 and acc = 0)
                            acc[k].x *= sc; acc[k].y *= sc; acc[k].z *= sc; acc[k].w *= sc; W[k] *= sc;
                            Mrow[k] = Mg;
                        }
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const bool on = ml[k][q].x != -INFINITY;
                            const float wgt = on ? exp2f(ml[k][q].x - Mrow[k]) : 0.f;
                            W[k] += wgt * ml[k][q].y;
                            acc[k].x += on ? wgt * v[k][q].x : 0.f; acc[k].y += on ? wgt * v[k][q].y : 0.f;
                            acc[k].z += on ? wgt * v[k][q].z : 0.f; acc[k].w += on ? wgt * v[k][q].w : 0.f;
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < RB; ++k) {
                    const int i = i0 + k * 8 * RW;
                    if (i >= n_mine) continue;
                    const int prow = r_begin + i;
                    const float inv = __fdividef(1.f, W[k]);
                    uint2 o2;
                    o2.x = pack_bf16(acc[k].x * inv, acc[k].y * inv);
                    o2.y = pack_bf16(acc[k].z * inv, acc[k].w * inv);
                    const int64_t grow = (int64_t)b.cu_new[s] + tok0 + prow;
                    const int c = (pch & ~7) | ((pch & 7) ^ (prow & 7));   // un-swizzle: which columns this chunk holds
                    *reinterpret_cast<uint2 *>((char *)a.out + (grow * g.Hq + h) * (D * 2) + c * 8) = o2;
                }
            }
        }
    }

    if (threadIdx.x == 128) { TL(33); TLG(61); }
    tc_fence_before();
    __syncthreads();
    if (warp == 2)
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tmem) : "memory");
}

}  // namespace

int sc_tc_tile_m() { return kPairM; }
int sc_tc_tile_n() { return kTN; }

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
static void fill_config(cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr, dim3 grid, int cluster, cudaStream_t st)
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
    cfg.attrs = attr;
    cfg.numAttrs = 1;
}

template <int D, int LEAN>
static cudaError_t launch_tc(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, dim3 grid, cudaStream_t st)
{
    cudaError_t e = prepare_tc<D, LEAN>();
    if (e != cudaSuccess) return e;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    fill_config<D, LEAN>(cfg, attr, grid, a.cluster_combine ? (int)grid.x : 1, st);
    return cudaLaunchKernelEx(&cfg, sc_attn_tc_kernel<D, LEAN>, g, b, a);
}

// CTAs that can be resident at once when the kernel is launched in clusters of `cluster` CTAs
// (each CTA needs a whole SM; a cluster must fit in one GPC).  0 if such clusters cannot launch.
template <int D, int LEAN>
static int wave_ctas(int cluster)
{
    if (prepare_tc<D, LEAN>() != cudaSuccess) return 0;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    fill_config<D, LEAN>(cfg, attr, dim3((unsigned)cluster, 1, 1), cluster, nullptr);
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
#ifdef SC_TC_PROBE
extern "C" int sc_probe_read(long long *host) { return (int)cudaMemcpyFromSymbol(host, sc_tl, sizeof(long long) * 256 * 64); }
#endif

cudaError_t sc_launch_attn_tc(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, cudaStream_t st)
{
    const int total_pairs = b.cu_mt[b.n_seq];
    if (total_pairs == 0) return cudaSuccess;
    dim3 grid((unsigned)a.n_splits, (unsigned)g.Hq, (unsigned)total_pairs);
#ifdef SC_TC_PROBE
    {
        const char *pf = getenv("SC_TC_PROBE");
        const int flags = pf ? atoi(pf) : 0;
        cudaMemcpyToSymbolAsync(sc_probe_flags, &flags, sizeof flags, 0, cudaMemcpyHostToDevice, st);
    }
#endif
    if (a.has_scat1)   // staged mode: a gather runs beside this kernel
        return g.D == 128 ? launch_tc<128, 1>(g, b, a, grid, st) : launch_tc<64, 1>(g, b, a, grid, st);
    return g.D == 128 ? launch_tc<128, 0>(g, b, a, grid, st) : launch_tc<64, 0>(g, b, a, grid, st);
}
