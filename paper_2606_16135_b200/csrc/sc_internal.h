// sc_internal.h -- shared between the translation units of libswiftcache.so.
// Not part of the public boundary (include/swiftcache.h is).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>
#include <mutex>
#include <vector>

#include "swiftcache.h"

// ----------------------------------------------------------------- geometry
struct ScGeom {
    int32_t L, Hq, Hkv, D, B;
    int32_t nh;           // D / 64: number of 128-byte halves per row
    int64_t chunk_bytes;  // B*D*2
    int64_t cell_bytes;   // 2*Hkv*chunk_bytes   (Eq. 1)
    int64_t block_bytes;  // L*cell_bytes        (block-major)
};

// Byte offset of (slot, d) inside a chunk: the 128B-swizzled K-major operand image
// (8-row x 128-byte atoms; 16-byte unit index XORed with the row index).
__host__ __device__ __forceinline__ uint32_t sc_chunk_off(int slot, int d, int nh)
{
    const int r = slot & 7, tg = slot >> 3, hf = d >> 6, c = (d & 63) >> 3;
    return (uint32_t)(tg * (nh * 1024) + hf * 1024 + r * 128 + ((c ^ r) << 4) + (d & 7) * 2);
}

// Where a kernel finds logical block j of sequence s.
struct ScKvView {
    char *base;             // pool_base + layer*cell_bytes, or an LSC buffer
    int64_t block_stride;   // block_bytes (pool) or cell_bytes (LSC)
    const int32_t *tables;  // DEVICE [n_seq][max_blocks]; nullptr => identity (LSC)
    int32_t max_blocks;
};

// A ragged batch, passed BY VALUE as a kernel parameter (no device descriptor copies).
struct ScBatch {
    int32_t n_seq;
    int32_t hist[SC_MAX_SEQS];        // T_h per sequence (or start_token for store/read)
    int32_t cu_new[SC_MAX_SEQS + 1];  // prefix sums of n_new
    int32_t lsc_off[SC_MAX_SEQS];     // first LSC block of each sequence
    int32_t cu_mt[SC_MAX_SEQS + 1];   // prefix sums of query M-tiles (engine specific)
    int32_t cu_blk[SC_MAX_SEQS + 1];  // prefix sums of blocks to copy (gather)
    int32_t rc_blk[SC_MAX_SEQS];      // leading logical blocks that are RESIDENT (regular cache): never gathered,
                                      // read in place through the table even in staged mode
    int32_t lsc_total;                // LSC blocks the whole batch occupies
};

__device__ __forceinline__ int64_t sc_phys_block(const ScKvView &v, const ScBatch &b, int s, int lb)
{
    return v.tables ? (int64_t)__ldg(v.tables + (int64_t)s * v.max_blocks + lb)
                    : (int64_t)(b.lsc_off[s] + lb);
}

// ------------------------------------------------------------------- pool
struct sc_pool {
    sc_pool_config_t cfg;
    ScGeom g;
    char *pool_base = nullptr;
    char *lsc_base = nullptr;
    int64_t pool_bytes = 0, lsc_buffer_bytes = 0;
    bool host_only = false;

    // allocator (a1): LIFO free list + state per block
    std::mutex mu;
    std::vector<int32_t> free_list;
    std::vector<uint8_t> allocated;

    // device scratch owned by the library
    char *scratch = nullptr;
    int64_t scratch_bytes = 0;
    float *part_o = nullptr;   // [max_splits][max_new_tokens][Hq][D] fp32, unnormalised
    float *part_ml = nullptr;  // [max_splits][max_new_tokens][Hq][2]  (m in log2 units, l)
    int32_t max_splits = 1;
    // host-io staging for sc_prefill_turn(io_kind = HOST_PINNED): 2 slots of q,k,v,out
    char *stage[2] = {nullptr, nullptr};
    int64_t stage_bytes = 0;

    int32_t attn_engine = SC_ENGINE_AUTO, copy_engine = SC_COPY_AUTO;
    int32_t split_tiles_override = 0;
    int32_t resident_blocks = 0;      // f3: leading blocks of every conversation kept as regular cache
    int32_t n_sms = 148;

    // pipeline resources (a8)
    cudaStream_t h2d_stream = nullptr, d2h_stream = nullptr;
    cudaEvent_t ev_load[2] = {nullptr, nullptr};   // load into LSC[b] finished
    cudaEvent_t ev_attn[2] = {nullptr, nullptr};   // attention reading LSC[b] finished
    cudaEvent_t ev_h2d[2] = {nullptr, nullptr};    // staging slot filled
    cudaEvent_t ev_comp[2] = {nullptr, nullptr};   // compute done with staging slot
    cudaEvent_t ev_d2h[2] = {nullptr, nullptr};    // out of staging slot copied back
    cudaEvent_t ev_fork = nullptr;

    int64_t launches = 0;

    // per-kernel timing (sc_profile_enable / sc_profile_collect)
    struct ProfRec { cudaEvent_t a, b; int kind; };
    bool profiling = false;
    std::vector<ProfRec> prof;
};

// Brackets one kernel launch with events on its own stream while profiling is on.
struct ScProfScope {
    sc_pool *p; cudaStream_t st; cudaEvent_t b = nullptr;
    ScProfScope(sc_pool *pool, int kind, cudaStream_t s) : p(pool), st(s)
    {
        if (!p->profiling) return;
        sc_pool::ProfRec r;
        r.kind = kind;
        if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) return;
        cudaEventRecord(r.a, st);
        b = r.b;
        p->prof.push_back(r);
    }
    ~ScProfScope() { if (b) cudaEventRecord(b, st); }
};

// error reporting (sc_api.cu): formats into the thread-local buffer of sc_last_error()
sc_status_t sc_fail(sc_status_t code, const char *fmt, ...);
sc_status_t sc_cuda_fail(cudaError_t e, const char *what);
const char *sc_err_buf();

// Function attributes (dynamic shared memory, cluster size) are per device: true the first
// time it is called for the calling thread's current device with this mask (up to 64 devices).
inline bool sc_first_use_on_device(std::atomic<uint64_t> &mask)
{
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev > 63) return true;   // just set it again
    const uint64_t bit = 1ull << dev;
    return (mask.fetch_or(bit) & bit) == 0;
}
constexpr int SC_MAX_DEVICES = 64;

// ------------------------------------------------------- kernel launchers
// sc_copy.cu
cudaError_t sc_launch_scatter(const ScGeom &g, const void *k, const void *v, const ScBatch &b,
                              const ScKvView &dst0, const ScKvView *dst1, bool pad_last_block, cudaStream_t st);
cudaError_t sc_launch_read(const ScGeom &g, void *k_out, void *v_out, const ScBatch &b,
                           const ScKvView &src, cudaStream_t st);
cudaError_t sc_launch_gather(const ScGeom &g, const ScBatch &b, const ScKvView &src,
                             const ScKvView &dst, int engine, int n_sms, cudaStream_t st);

// sc_attn_mma.cu  (mma.sync engine) and the split-KV combine
struct ScAttnArgs {
    const void *q;      // [sum n][Hq][D] bf16
    void *out;          // [sum n][Hq][D] bf16
    ScKvView kv;        // history + new tokens, through the table (or LSC identity)
    ScKvView kv_res;    // staged mode with a regular cache: where logical blocks < rc_blk[s] are read (the pool)
    int32_t has_res;
    float *part_o, *part_ml;
    int32_t part_half;    // the O partials are fp16 rows scaled by a power of two (tcgen05 engine), else fp32
    // tcgen05 engine: the scatter of the new K/V (a5) is folded into the attention kernel
    const void *k_new, *v_new;   // [sum n][Hkv][D] bf16, or nullptr: already scattered
    ScKvView scat0, scat1;       // where to scatter: the pool, and (staged mode) the LSC
    int32_t has_scat1;
    int32_t cluster_combine;  // tcgen05 engine: the splits of a query tile group form a cluster and merge in kernel
    int32_t pdl;          // tcgen05 engine: launch with programmatic stream serialization
    int32_t split_units;  // KV units per split; a unit is the engine's split granule in tokens
                          // (sc_mma_split_unit(): its 64-token tile; sc_tc_split_unit(): a 16-token pool block)
    int32_t n_splits;     // grid extent over splits (max over rows)
    int32_t total_new;    // sum n
};
int sc_mma_tile_m();       // query rows per CTA of the mma.sync engine
int sc_mma_split_unit();   // tokens per split unit (its KV tile)
cudaError_t sc_launch_attn_mma(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, cudaStream_t st);
// sc_attn_tc.cu  (tcgen05 / TMEM engine): a CTA owns a pair of 128-row query tiles
int sc_tc_tile_m();
int sc_tc_split_unit();    // tokens per split unit (a pool block)
int sc_tc_max_cluster();   // most splits the in-kernel (cluster) combine handles
int sc_tc_wave_ctas(int D, int lean, int cluster);   // co-resident CTAs when launched in clusters of that size
cudaError_t sc_launch_attn_tc(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, cudaStream_t st);
// sc_attn_decode.cu  (decode engine): one CTA per (split, KV head, conversation), at most 16 rows
int sc_dec_max_rows();     // (new token, query head of the group) rows a CTA holds
int sc_dec_split_unit();   // tokens per split unit (its 64-token tile)
int sc_dec_ctas_per_sm();
cudaError_t sc_launch_attn_decode(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, cudaStream_t st);
cudaError_t sc_launch_combine(const ScGeom &g, const ScBatch &b, const ScAttnArgs &a, int tile_m,
                              int split_unit, cudaStream_t st);
