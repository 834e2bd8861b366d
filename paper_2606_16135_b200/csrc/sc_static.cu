// sc_static.cu -- sc_prefill_layer_static: one layer of prefill (a5 scatter, a6 attention, a7 split-KV
// merge) for callers that are not allowed to allocate device memory.
//
// Who that is.  In the paper's deployment the KV pool is *donated* memory: a worker hands every
// byte of HBM it can spare to the block pool, and the elastic resize of
// Sec. 3.4 keeps it that way.  A serving process in that state has nothing left for cudaMalloc to
// give out, so sc_pool_create's scratch allocation may simply fail.  And a process in the middle of
// serving cannot afford the call even when it would succeed: cudaMalloc and cudaFree wait for the
// whole device, i.e. they stall every stream of every model on the GPU.  The regular path needs a
// pool object (which allocates its split-KV scratch, streams and events); this file is the way
// round it: no pool object, and the scratch the split-KV attention needs is part of the library
// image itself.
//
// How.  The partial (m, l, O) triples that the split attention CTAs write and the merge kernel reads
// live in sc_static_scratch below, a file-scope __device__ array of SC_STATIC_SCRATCH_BYTES.  The
// driver gives every GPU that loads libswiftcache.so its own copy when the module is loaded and
// keeps it until the process exits.  The kernels are the ones the regular path launches
// (sc_attn_mma.cu, sc_copy.cu); only the place the partials go differs, so for the same partition
// the output is bit-identical to sc_prefill_layer(FUSED) with the mma.sync engine.
//
// Rules a reader of this file should know:
//   - In HOST code `sc_static_scratch` is not a device address; it is a host-side shadow the runtime
//     uses to look the real one up.  The address a kernel may be given comes from
//     cudaGetSymbolAddress, asked once per device with that device current (scratch_on_this_device).
//   - One array per GPU, shared by every call and every stream: two calls whose kernels may run at
//     the same time on one GPU overwrite each other's partials.  Callers serialise them.
//   - The array keeps what the previous call left.  Nothing in it has to start at zero: the merge
//     reads only partials that the attention kernel of the SAME call has written (a partition that
//     holds no key of a query tile is neither written nor read), so no clear is enqueued.
//   - No cudaMalloc, cudaFree, stream / event creation or other allocating routine is called here.
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>

#include "sc_internal.h"

// 256-byte aligned so the fp32 partial rows keep the 16-byte alignment the vector accesses need.
static __device__ __align__(256) unsigned char sc_static_scratch[SC_STATIC_SCRATCH_BYTES];

namespace {

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

struct PerDevice {
    unsigned char *scratch = nullptr;   // the device address of sc_static_scratch on that GPU
    int n_sms = 0;
};
std::mutex g_mu;
PerDevice g_dev[SC_MAX_DEVICES];

// First call on a GPU: resolve the symbol for the CURRENT device, remember it.  A failure is not
// remembered, the next call tries again.
sc_status_t scratch_on_this_device(PerDevice *out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return sc_cuda_fail(e, "cudaGetDevice");
    if (dev < 0 || dev >= SC_MAX_DEVICES) return sc_fail(SC_ERR_UNSUPPORTED, "device ordinal %d >= %d", dev, SC_MAX_DEVICES);
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_dev[dev].scratch) {
        unsigned char *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, sc_static_scratch);
        if (e != cudaSuccess) return sc_cuda_fail(e, "cudaGetSymbolAddress(sc_static_scratch)");
        if (!ptr || ((uintptr_t)ptr & 255)) return sc_fail(SC_ERR_CUDA, "static scratch resolved to %p", (void *)ptr);
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return sc_cuda_fail(e, "cudaDeviceGetAttribute");
        g_dev[dev].n_sms = sms;
        g_dev[dev].scratch = ptr;
    }
    *out = g_dev[dev];
    return SC_OK;
}

// bytes of the partials of n_splits partitions: O rows fp32, then (m, l) pairs, the second part
// starting on a 256-byte boundary
inline int64_t part_o_bytes(int64_t n_splits, int64_t rows, int D) { return (n_splits * rows * D * 4 + 255) & ~(int64_t)255; }
inline int64_t partial_bytes(int64_t n_splits, int64_t rows, int D) { return part_o_bytes(n_splits, rows, D) + n_splits * rows * 2 * 4; }

}  // namespace

extern "C" sc_status_t sc_prefill_layer_static(const sc_pool_config_t *cfg, void *pool_base, int32_t layer,
                                               const void *q, const void *k_new, const void *v_new,
                                               const int32_t *table_dev, int32_t n_table, int32_t hist_len,
                                               int32_t n_new, int32_t tiles_per_split, void *out, void *stream)
{
    // ---- host-side checks; nothing has touched the device yet
    if (!cfg) return sc_fail(SC_ERR_INVALID_ARG, "config is NULL");
    if (cfg->n_layers <= 0 || cfg->n_q_heads <= 0 || cfg->n_kv_heads <= 0)
        return sc_fail(SC_ERR_INVALID_ARG, "non-positive size in config");
    if (cfg->head_dim != 64 && cfg->head_dim != 128) return sc_fail(SC_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", cfg->head_dim);
    if (cfg->block_size != 16) return sc_fail(SC_ERR_UNSUPPORTED, "block_size %d != 16", cfg->block_size);
    if (cfg->n_q_heads % cfg->n_kv_heads)
        return sc_fail(SC_ERR_UNSUPPORTED, "n_q_heads %d not a multiple of n_kv_heads %d", cfg->n_q_heads, cfg->n_kv_heads);
    if (layer < 0 || layer >= cfg->n_layers) return sc_fail(SC_ERR_INVALID_ARG, "layer %d not in [0,%d)", layer, cfg->n_layers);
    if (hist_len < 0 || n_new < 0 || tiles_per_split < 0) return sc_fail(SC_ERR_INVALID_ARG, "negative length");
    if (n_new == 0) return SC_OK;
    if (!pool_base || !q || !out || !table_dev || n_table <= 0) return sc_fail(SC_ERR_INVALID_ARG, "NULL tensor or table");
    if ((k_new == nullptr) != (v_new == nullptr)) return sc_fail(SC_ERR_INVALID_ARG, "k_new and v_new must both be given or both be NULL");
    if ((uintptr_t)pool_base & 1023) return sc_fail(SC_ERR_INVALID_ARG, "pool_base must be 1024-byte aligned");
    const int64_t tot = (int64_t)hist_len + n_new;
    if (tot > (int64_t)n_table * cfg->block_size)
        return sc_fail(SC_ERR_CAPACITY, "%lld tokens exceed table of %d blocks", (long long)tot, n_table);

    ScGeom g;
    g.L = cfg->n_layers; g.Hq = cfg->n_q_heads; g.Hkv = cfg->n_kv_heads; g.D = cfg->head_dim;
    g.B = cfg->block_size; g.nh = g.D / 64;
    g.chunk_bytes = (int64_t)g.B * g.D * 2;
    g.cell_bytes = 2 * (int64_t)g.Hkv * g.chunk_bytes;      // Eq. 1
    g.block_bytes = (int64_t)g.L * g.cell_bytes;            // block-major

    // ---- partition of the keys [0, hist_len + n_new), in the 64-token tiles of the mma.sync engine
    const int tile_m = sc_mma_tile_m(), unit = sc_mma_split_unit();
    const int max_units = std::max(1, ceil_div((int)tot, unit));
    const int64_t rows = (int64_t)n_new * g.Hq;
    const int max_partitions = 32;                           // the merge keeps one partition per lane
    int split_units, n_splits;
    const bool forced = tiles_per_split > 0;
    if (forced) {
        split_units = tiles_per_split;
        if (ceil_div(max_units, split_units) > max_partitions) split_units = ceil_div(max_units, max_partitions);
        n_splits = ceil_div(max_units, split_units);
        if (n_splits > 1 && partial_bytes(n_splits, rows, g.D) > (int64_t)SC_STATIC_SCRATCH_BYTES)
            return sc_fail(SC_ERR_CAPACITY,
                           "%d partitions x %d new tokens x %d heads x D %d need %lld bytes of partials; the static "
                           "scratch holds SC_STATIC_SCRATCH_BYTES = %lld (use fewer partitions, or 0 = automatic)",
                           n_splits, n_new, g.Hq, g.D, (long long)partial_bytes(n_splits, rows, g.D),
                           (long long)SC_STATIC_SCRATCH_BYTES);
    }

    // ---- set-up (first call on this GPU): where the scratch is
    PerDevice pd;
    sc_status_t st = scratch_on_this_device(&pd);
    if (st) return st;

    if (!forced) {
        // enough CTAs for about three per SM (what the kernel's registers and shared memory allow),
        // but never more partitions than fit in the array; one partition needs no scratch at all
        const int64_t ctas1 = (int64_t)g.Hq * ceil_div(n_new, tile_m);
        int want = (int)std::min<int64_t>(max_partitions, (3LL * pd.n_sms + ctas1 - 1) / ctas1);
        want = std::max(1, std::min(want, max_units));
        while (want > 1 && partial_bytes(want, rows, g.D) > (int64_t)SC_STATIC_SCRATCH_BYTES) --want;
        split_units = ceil_div(max_units, want);
        n_splits = ceil_div(max_units, split_units);
    }

    ScBatch b;
    memset(&b, 0, sizeof b);
    b.n_seq = 1;
    b.hist[0] = hist_len;
    b.cu_new[1] = n_new;
    b.cu_mt[1] = ceil_div(n_new, tile_m);
    b.cu_blk[1] = ceil_div(hist_len, g.B);
    b.lsc_total = ceil_div((int)tot, g.B);

    ScKvView pv;
    pv.base = (char *)pool_base + (int64_t)layer * g.cell_bytes;
    pv.block_stride = g.block_bytes;
    pv.tables = table_dev;
    pv.max_blocks = n_table;

    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    // 1. scatter of the new K/V into the pool blocks, rest of the last block set to zero (a5)
    if (k_new) {
        e = sc_launch_scatter(g, k_new, v_new, b, pv, nullptr, true, s);
        if (e != cudaSuccess) return sc_cuda_fail(e, "scatter launch");
    }
    // 2. attention over the pool blocks in place (a6); partials into the static array
    ScAttnArgs a;
    memset(&a, 0, sizeof a);
    a.q = q;
    a.out = out;
    a.kv = pv;
    a.kv_res = pv;
    a.scat0 = pv;
    a.scat1 = pv;
    a.part_o = (float *)pd.scratch;
    a.part_ml = (float *)(pd.scratch + part_o_bytes(n_splits, rows, g.D));
    a.part_half = 0;
    a.split_units = split_units;
    a.n_splits = n_splits;
    a.total_new = n_new;
    e = sc_launch_attn_mma(g, b, a, s);
    if (e != cudaSuccess) return sc_cuda_fail(e, "attention launch");
    // 3. merge of the partitions (a7)
    if (n_splits > 1) {
        e = sc_launch_combine(g, b, a, tile_m, unit, s);
        if (e != cudaSuccess) return sc_cuda_fail(e, "merge launch");
    }
    return SC_OK;
}
