// sc_ops.cu -- the data calls of the C ABI (a3-a9): argument checking on the host,
// then kernel launches on the caller's stream.  No step of the path runs on the CPU.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "sc_internal.h"

namespace {

#define SC_CUDA(call)                                                   \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return sc_cuda_fail(e_, #call);          \
    } while (0)

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

sc_status_t check_pool(sc_pool_t *p, int32_t layer)
{
    if (!p) return sc_fail(SC_ERR_INVALID_ARG, "pool is NULL");
    if (p->host_only) return sc_fail(SC_ERR_CUDA, "host-only pool (created without memory): no data calls");
    if (layer < 0 || layer >= p->g.L) return sc_fail(SC_ERR_INVALID_ARG, "layer %d not in [0,%d)", layer, p->g.L);
    return SC_OK;
}

ScKvView pool_view(const sc_pool_t *p, int layer, const int32_t *tables, int max_blocks)
{
    ScKvView v;
    v.base = p->pool_base + (int64_t)layer * p->g.cell_bytes;
    v.block_stride = p->g.block_bytes;
    v.tables = tables;
    v.max_blocks = max_blocks;
    return v;
}

ScKvView lsc_view(const sc_pool_t *p, int buf)
{
    ScKvView v;
    v.base = p->lsc_base + (int64_t)buf * p->lsc_buffer_bytes;
    v.block_stride = p->g.cell_bytes;
    v.tables = nullptr;
    v.max_blocks = 0;
    return v;
}

// Validates a ragged batch and fills the by-value descriptor.  `with_new` = 0 for the
// gather (blocks to copy = ceil(hist/B)), but LSC offsets always reserve room for the
// new tokens so load and prefill agree on the placement.
sc_status_t make_batch(const sc_pool_t *p, int n_seq, const int32_t *hist_lens, const int32_t *cu_new,
                       int max_blocks, int tile_m, ScBatch *b)
{
    if (n_seq <= 0 || n_seq > p->cfg.max_seqs) return sc_fail(SC_ERR_CAPACITY, "n_seq %d not in [1,%d]", n_seq, p->cfg.max_seqs);
    if (!hist_lens || !cu_new) return sc_fail(SC_ERR_INVALID_ARG, "hist_lens / cu_new is NULL");
    if (cu_new[0] != 0) return sc_fail(SC_ERR_INVALID_ARG, "cu_new[0] != 0");
    memset(b, 0, sizeof *b);
    b->n_seq = n_seq;
    int lsc = 0, mt = 0, blk = 0;
    for (int s = 0; s < n_seq; ++s) {
        const int n = cu_new[s + 1] - cu_new[s];
        if (hist_lens[s] < 0 || n < 0) return sc_fail(SC_ERR_INVALID_ARG, "negative length in sequence %d", s);
        const int64_t tot = (int64_t)hist_lens[s] + n;
        if (tot > (int64_t)max_blocks * p->g.B)
            return sc_fail(SC_ERR_CAPACITY, "sequence %d: %lld tokens exceed table of %d blocks", s, (long long)tot, max_blocks);
        b->hist[s] = hist_lens[s];
        b->cu_new[s] = cu_new[s];
        b->lsc_off[s] = lsc;
        b->cu_mt[s] = mt;
        b->cu_blk[s] = blk;
        b->rc_blk[s] = std::min(p->resident_blocks, hist_lens[s] / p->g.B);   // complete history blocks only
        lsc += ceil_div((int)tot, p->g.B);
        mt += ceil_div(n, tile_m);
        blk += ceil_div(hist_lens[s], p->g.B) - b->rc_blk[s];
    }
    b->cu_new[n_seq] = cu_new[n_seq];
    b->cu_mt[n_seq] = mt;
    b->cu_blk[n_seq] = blk;
    b->lsc_total = lsc;
    if (cu_new[n_seq] > p->cfg.max_new_tokens)
        return sc_fail(SC_ERR_CAPACITY, "%d new tokens > max_new_tokens %d", cu_new[n_seq], p->cfg.max_new_tokens);
    return SC_OK;
}

int lsc_blocks_needed(const ScBatch &b) { return b.lsc_total; }

// How the KV range of a batch is split over CTAs.  Splits are counted in the engine's split unit
// (tcgen05: a 16-token pool block, so that e.g. 336 blocks over 4 CTAs are 84 each = 10.5 KV tiles;
// mma.sync: its 64-token tile).  Every (query tile group, head) needs ceil(units/split) CTAs; the
// grid runs in waves, and a CTA costs its KV tiles plus a fixed overhead (prologue, epilogue).
// Costs are in units of one 128-token KV tile (~1.8 us on B200), fitted to measurements:
//   cluster (tcgen05, <= 16 splits, ONE wave only -- clusters of whole-SM CTAs place badly over
//            several waves -- and <= 128 tiles per CTA): in-kernel scatter + DSMEM combine, ~3
//   plain  : separate scatter (~5) and combine (~1.3 per split) kernels, partial write ~2 per wave
// Depends on logical lengths only.
struct SplitChoice { int split_units; bool cluster; };

SplitChoice choose_split(const sc_pool_t *p, int n_seq, const int32_t *hist_lens, const int32_t *cu_new,
                         int tile_m, int unit, bool tc, bool staged)
{
    int max_units = 1;
    for (int i = 0; i < n_seq; ++i)
        max_units = std::max(max_units, ceil_div(hist_lens[i] + (cu_new[i + 1] - cu_new[i]), unit));
    const double units_per_tile = 128.0 / unit;
    SplitChoice best = {max_units, false};
    double best_cost = 1e30;
    for (int n_sp = 1; n_sp <= p->max_splits; ++n_sp) {
        const int split = ceil_div(max_units, n_sp);
        if (n_sp > 1 && ceil_div(max_units, split) != n_sp) continue;     // same split as a smaller n_sp
        int64_t ctas = 0;
        for (int i = 0; i < n_seq; ++i) {
            const int n = cu_new[i + 1] - cu_new[i];
            for (int mt = 0; mt * tile_m < n; ++mt) {
                const int kmax = hist_lens[i] + std::min(n, (mt + 1) * tile_m);
                ctas += (int64_t)p->g.Hq * ceil_div(ceil_div(kmax, unit), split);
            }
        }
        for (int use_cluster = 0; use_cluster < 2; ++use_cluster) {
            int64_t wave = (int64_t)p->n_sms * (tc ? 1 : 3);
            double extra = 0.0;
            if (use_cluster) {
                if (!tc || n_sp < 2 || n_sp > sc_tc_max_cluster() || split > 128 * units_per_tile) continue;
                wave = sc_tc_wave_ctas(p->g.D, staged, n_sp);
                // the launch is n_sp CTAs per (pair, head) whether or not a sequence needs them all
                int64_t launched = 0;
                for (int i = 0; i < n_seq; ++i)
                    launched += (int64_t)p->g.Hq * ceil_div(cu_new[i + 1] - cu_new[i], tile_m) * n_sp;
                if (wave <= 0 || launched > wave) continue;
                extra = 3.0;
            }
            const double waves = (double)((ctas + wave - 1) / wave);
            if (!use_cluster && n_sp > 1) extra = (tc ? 5.0 : 0.5) + 1.3 * n_sp + 2.0 * waves;
            const double cost = waves * (split / units_per_tile + 3.0) + extra;
            if (cost < best_cost - 1e-9) { best_cost = cost; best = {split, use_cluster != 0}; }
        }
    }
    best.split_units = std::max(best.split_units, 1);
    return best;
}

}  // namespace

extern "C" {

sc_status_t sc_store_prefix(sc_pool_t *pool, int32_t layer, const void *k, const void *v,
                            int32_t start_token, int32_t n_tokens, const int32_t *table_dev,
                            int32_t n_table, void *stream)
{
    sc_status_t st = check_pool(pool, layer);
    if (st) return st;
    if (start_token < 0 || n_tokens < 0) return sc_fail(SC_ERR_INVALID_ARG, "negative token range");
    if (n_tokens == 0) return SC_OK;
    if (!k || !v || !table_dev) return sc_fail(SC_ERR_INVALID_ARG, "NULL tensor or table");
    if ((int64_t)start_token + n_tokens > (int64_t)n_table * pool->g.B)
        return sc_fail(SC_ERR_CAPACITY, "tokens [%d,%d) exceed table of %d blocks", start_token,
                       start_token + n_tokens, n_table);
    ScBatch b;
    memset(&b, 0, sizeof b);
    b.n_seq = 1;
    b.hist[0] = start_token;
    b.cu_new[1] = n_tokens;
    {
        ScProfScope ps(pool, SC_KERNEL_SCATTER, (cudaStream_t)stream);
        SC_CUDA(sc_launch_scatter(pool->g, k, v, b, pool_view(pool, layer, table_dev, n_table), nullptr, false,
                                  (cudaStream_t)stream));
    }
    pool->launches += 1;
    return SC_OK;
}

sc_status_t sc_read_tokens(sc_pool_t *pool, int32_t layer, int32_t src, const int32_t *table_dev,
                           int32_t n_table, int32_t lsc_block_off, int32_t start_token,
                           int32_t n_tokens, void *k_out, void *v_out, void *stream)
{
    sc_status_t st = check_pool(pool, layer);
    if (st) return st;
    if (start_token < 0 || n_tokens < 0 || src < 0 || src > 2) return sc_fail(SC_ERR_INVALID_ARG, "bad range or src");
    if (n_tokens == 0) return SC_OK;
    if (!k_out || !v_out) return sc_fail(SC_ERR_INVALID_ARG, "NULL output");
    ScBatch b;
    memset(&b, 0, sizeof b);
    b.n_seq = 1;
    b.hist[0] = start_token;
    b.cu_new[1] = n_tokens;
    ScKvView view;
    if (src == 0) {
        if (!table_dev) return sc_fail(SC_ERR_INVALID_ARG, "table is NULL");
        if ((int64_t)start_token + n_tokens > (int64_t)n_table * pool->g.B)
            return sc_fail(SC_ERR_CAPACITY, "tokens exceed table of %d blocks", n_table);
        view = pool_view(pool, layer, table_dev, n_table);
    } else {
        if (!pool->lsc_base) return sc_fail(SC_ERR_CAPACITY, "pool has no LSC");
        const int last = lsc_block_off + ceil_div(start_token + n_tokens, pool->g.B);
        if (lsc_block_off < 0 || last > pool->cfg.lsc_blocks)
            return sc_fail(SC_ERR_CAPACITY, "tokens exceed the LSC (%d blocks)", pool->cfg.lsc_blocks);
        view = lsc_view(pool, src - 1);
        b.lsc_off[0] = lsc_block_off;
    }
    SC_CUDA(sc_launch_read(pool->g, k_out, v_out, b, view, (cudaStream_t)stream));
    pool->launches += 1;
    return SC_OK;
}

sc_status_t sc_load_layer_batched(sc_pool_t *pool, int32_t layer, const int32_t *tables_dev,
                                  int32_t max_blocks, int32_t n_seq, const int32_t *hist_lens,
                                  const int32_t *cu_new, int32_t buf, void *stream)
{
    sc_status_t st = check_pool(pool, layer);
    if (st) return st;
    if (!tables_dev || max_blocks <= 0) return sc_fail(SC_ERR_INVALID_ARG, "bad table");
    if (buf < 0 || buf > 1) return sc_fail(SC_ERR_INVALID_ARG, "buf %d not in {0,1}", buf);
    ScBatch b;
    st = make_batch(pool, n_seq, hist_lens, cu_new, max_blocks, sc_mma_tile_m(), &b);
    if (st) return st;
    if (!pool->lsc_base || lsc_blocks_needed(b) > pool->cfg.lsc_blocks)
        return sc_fail(SC_ERR_CAPACITY, "batch needs %d LSC blocks, buffer holds %d", lsc_blocks_needed(b),
                       pool->cfg.lsc_blocks);
    int engine = pool->copy_engine;
    if (engine == SC_COPY_AUTO) engine = SC_COPY_LDG;
    {
        ScProfScope ps(pool, SC_KERNEL_GATHER, (cudaStream_t)stream);
        SC_CUDA(sc_launch_gather(pool->g, b, pool_view(pool, layer, tables_dev, max_blocks), lsc_view(pool, buf),
                                 engine, pool->n_sms, (cudaStream_t)stream));
    }
    pool->launches += (b.cu_blk[n_seq] > 0);
    return SC_OK;
}

sc_status_t sc_load_layer(sc_pool_t *pool, int32_t layer, const int32_t *table_dev, int32_t n_table,
                          int32_t hist_len, int32_t buf, void *stream)
{
    // reserve nothing for new tokens here: the single-sequence LSC always starts at block 0
    const int32_t cu[2] = {0, 0};
    if (pool && hist_len > (int64_t)n_table * pool->g.B)
        return sc_fail(SC_ERR_CAPACITY, "hist_len %d exceeds table of %d blocks", hist_len, n_table);
    return sc_load_layer_batched(pool, layer, table_dev, n_table, 1, &hist_len, cu, buf, stream);
}

sc_status_t sc_prefill_layer_batched(sc_pool_t *pool, int32_t layer, const void *q, const void *k_new,
                                     const void *v_new, const int32_t *tables_dev, int32_t max_blocks,
                                     int32_t n_seq, const int32_t *hist_lens, const int32_t *cu_new,
                                     int32_t buf, int32_t mode, void *out, void *stream)
{
    sc_status_t st = check_pool(pool, layer);
    if (st) return st;
    if (!q || !k_new || !v_new || !out || !tables_dev || max_blocks <= 0)
        return sc_fail(SC_ERR_INVALID_ARG, "NULL tensor or table");
    if (mode != SC_ATTN_STAGED && mode != SC_ATTN_FUSED) return sc_fail(SC_ERR_INVALID_ARG, "mode %d", mode);
    if (buf < 0 || buf > 1) return sc_fail(SC_ERR_INVALID_ARG, "buf %d not in {0,1}", buf);
    int engine = pool->attn_engine;
    // A few new tokens per conversation (decode): all rows of a KV head's group fit one 16-row CTA of
    // the decode engine, which is built for the paged read that is left (sc_attn_decode.cu).
    bool dec_fits = n_seq > 0 && hist_lens && cu_new;
    for (int i = 0; dec_fits && i < n_seq; ++i)
        dec_fits = (int64_t)(cu_new[i + 1] - cu_new[i]) * (pool->g.Hq / pool->g.Hkv) <= sc_dec_max_rows();
    if (engine == SC_ENGINE_DECODE && !dec_fits)
        return sc_fail(SC_ERR_UNSUPPORTED, "decode engine: more than %d (new token, query head) rows per KV head",
                       sc_dec_max_rows());
    if (engine == SC_ENGINE_AUTO) {
        // The decode engine costs two more launches per layer (scatter, merge) than the tcgen05 kernel with
        // its folded scatter and cluster merge, and reads the KV faster: measured cross-over at ~8k tokens
        // x 32 KV heads x D 128 (27.5 vs 32 us per layer at 5 120 tokens, 194 vs 135 us at 50 000).
        int64_t kv_bytes = 0;
        for (int i = 0; dec_fits && i < n_seq; ++i)
            kv_bytes += ((int64_t)hist_lens[i] + (cu_new[i + 1] - cu_new[i])) * pool->g.Hkv * pool->g.D * 4;
        const bool long_enough = kv_bytes >= ((int64_t)128 << 20);
        engine = (dec_fits && long_enough && !(mode == SC_ATTN_STAGED && pool->resident_blocks > 0))
                     ? SC_ENGINE_DECODE : SC_ENGINE_TCGEN05;
    }
    const bool tc = (engine == SC_ENGINE_TCGEN05), dec = (engine == SC_ENGINE_DECODE);
    const int tile_m = tc ? sc_tc_tile_m() : dec ? sc_dec_max_rows() : sc_mma_tile_m();
    const int unit = tc ? sc_tc_split_unit() : dec ? sc_dec_split_unit() : sc_mma_split_unit();
    ScBatch b;
    st = make_batch(pool, n_seq, hist_lens, cu_new, max_blocks, tile_m, &b);
    if (st) return st;
    const int total_new = b.cu_new[n_seq];
    if (total_new == 0) return SC_OK;
    const bool staged = (mode == SC_ATTN_STAGED);
    if (staged && (!pool->lsc_base || lsc_blocks_needed(b) > pool->cfg.lsc_blocks))
        return sc_fail(SC_ERR_CAPACITY, "batch needs %d LSC blocks, buffer holds %d", lsc_blocks_needed(b),
                       pool->cfg.lsc_blocks);
    const bool has_res = staged && pool->resident_blocks > 0;
    if (has_res && !tc)          // checked before the first launch: an error leaves pool and LSC untouched
        return sc_fail(SC_ERR_UNSUPPORTED, "resident blocks in staged mode need the tcgen05 engine");
    cudaStream_t s = (cudaStream_t)stream;
    const ScKvView pv = pool_view(pool, layer, tables_dev, max_blocks);
    const ScKvView lv = staged ? lsc_view(pool, buf) : pv;

    // split of the KV range over CTAs, when that is needed to fill the machine
    bool cluster = false;
    int max_units = 1;
    for (int i = 0; i < n_seq; ++i)
        max_units = std::max(max_units, ceil_div(hist_lens[i] + (cu_new[i + 1] - cu_new[i]), unit));
    int split_units;
    if (dec && pool->split_tiles_override <= 0) {
        // one wave: as many splits as fill every CTA slot of the GPU once
        const int slots = pool->n_sms * sc_dec_ctas_per_sm(), per_split = pool->g.Hkv * n_seq;
        const int n_sp = std::max(1, std::min(std::min(slots / per_split, pool->max_splits), max_units));
        split_units = ceil_div(max_units, n_sp);
    } else if (pool->split_tiles_override <= 0) {
        const SplitChoice c = choose_split(pool, n_seq, hist_lens, cu_new, tile_m, unit, tc, staged);
        split_units = c.split_units;
        cluster = c.cluster;
    } else {
        // forced split (tests, experiments), given in KV tiles of the engine (tcgen05: 128 tokens,
        // mma.sync: 64): cluster whenever such a cluster can be placed
        split_units = pool->split_tiles_override * (tc ? 128 / unit : 1);
        const int ns = ceil_div(max_units, split_units);
        cluster = tc && ns > 1 && ns <= sc_tc_max_cluster() && sc_tc_wave_ctas(pool->g.D, staged, ns) > 0;
    }
    int n_splits = ceil_div(max_units, split_units);
    if (n_splits > pool->max_splits) {
        split_units = ceil_div(max_units, pool->max_splits);
        n_splits = ceil_div(max_units, split_units);
        cluster = false;
    }
    if (n_splits == 1) cluster = false;
    // 1. scatter (a5): pool, and the LSC tail in staged mode.  The tcgen05 engine does it inside
    //    the attention kernel when a query pair's CTAs form a cluster (they share the work) or
    //    when there is a single CTA per pair -- but only where that makes ONE writer per row: no
    //    grouped-query heads (the query heads of a group would each store the KV head's rows) and
    //    one query pair per sequence (a later pair reads, and would store, the earlier pairs' rows).
    //    Otherwise the scatter kernel runs first; it too writes every row once.
    bool one_pair = true;
    for (int i = 0; i < n_seq; ++i) one_pair = one_pair && (cu_new[i + 1] - cu_new[i] <= tile_m);
    const bool fold_scatter = tc && (cluster || n_splits == 1) && pool->g.Hq == pool->g.Hkv && one_pair;
    if (!fold_scatter) {
        ScProfScope ps(pool, SC_KERNEL_SCATTER, s);
        SC_CUDA(sc_launch_scatter(pool->g, k_new, v_new, b, pv, staged ? &lv : nullptr, true, s));
        pool->launches += 1;
    }

    // 2. attention (a6)
    ScAttnArgs a;
    a.q = q;
    a.out = out;
    a.kv = lv;
    a.part_o = pool->part_o;
    a.part_ml = pool->part_ml;
    a.part_half = tc ? 1 : 0;
    a.k_new = fold_scatter ? k_new : nullptr;
    a.v_new = fold_scatter ? v_new : nullptr;
    a.kv_res = pv;
    a.has_res = has_res ? 1 : 0;
    a.scat0 = pv;
    a.scat1 = lv;
    a.has_scat1 = staged ? 1 : 0;
    a.cluster_combine = cluster ? 1 : 0;
    // programmatic dependent launch only in fused mode: in staged mode the early CTAs of the next layer
    // would sit on SMs that the concurrent gather of the copy stream can use in full
    a.pdl = (tc && !staged) ? 1 : 0;
    a.split_units = split_units;
    a.n_splits = n_splits;
    a.total_new = total_new;
    {
        ScProfScope ps(pool, SC_KERNEL_ATTENTION, s);
        SC_CUDA(tc ? sc_launch_attn_tc(pool->g, b, a, s)
                   : dec ? sc_launch_attn_decode(pool->g, b, a, s) : sc_launch_attn_mma(pool->g, b, a, s));
    }
    pool->launches += 1;
    // 3. combine (a7): with up to 16 splits in one wave the tcgen05 engine merges the partials itself
    //    (the splits of a query tile group form a thread-block cluster); otherwise a separate kernel
    if (n_splits > 1 && !a.cluster_combine) {
        {
            ScProfScope ps(pool, SC_KERNEL_COMBINE, s);
            SC_CUDA(sc_launch_combine(pool->g, b, a, tile_m, unit, s));
        }
        pool->launches += 1;
    }
    return SC_OK;
}

sc_status_t sc_prefill_layer(sc_pool_t *pool, int32_t layer, const void *q, const void *k_new,
                             const void *v_new, const int32_t *table_dev, int32_t n_table,
                             int32_t hist_len, int32_t n_new, int32_t buf, int32_t mode, void *out,
                             void *stream)
{
    if (n_new < 0) return sc_fail(SC_ERR_INVALID_ARG, "n_new < 0");
    const int32_t cu[2] = {0, n_new};
    return sc_prefill_layer_batched(pool, layer, q, k_new, v_new, table_dev, n_table, 1, &hist_len, cu,
                                    buf, mode, out, stream);
}

sc_status_t sc_prefill_turn(sc_pool_t *pool, const void *q_all, const void *k_all, const void *v_all,
                            void *out_all, int32_t io_kind, const int32_t *tables_dev,
                            int32_t max_blocks, int32_t n_seq, const int32_t *hist_lens,
                            const int32_t *cu_new, int32_t mode, void *copy_stream, void *compute_stream)
{
    return sc_prefill_turn_ex(pool, q_all, k_all, v_all, out_all, io_kind, tables_dev, max_blocks, n_seq, hist_lens,
                              cu_new, mode, copy_stream, compute_stream, nullptr);
}

sc_status_t sc_prefill_turn_ex(sc_pool_t *pool, const void *q_all, const void *k_all, const void *v_all,
                               void *out_all, int32_t io_kind, const int32_t *tables_dev,
                               int32_t max_blocks, int32_t n_seq, const int32_t *hist_lens,
                               const int32_t *cu_new, int32_t mode, void *copy_stream, void *compute_stream,
                               const sc_turn_options_t *opt)
{
    sc_status_t st = check_pool(pool, 0);
    if (st) return st;
    const int nbuf = opt ? opt->lsc_buffers : 2;
    if (nbuf != 1 && nbuf != 2) return sc_fail(SC_ERR_INVALID_ARG, "lsc_buffers %d not in {1,2}", nbuf);
    if (!q_all || !k_all || !v_all || !out_all) return sc_fail(SC_ERR_INVALID_ARG, "NULL tensor");
    if (io_kind != SC_MEM_DEVICE && io_kind != SC_MEM_HOST_PINNED) return sc_fail(SC_ERR_INVALID_ARG, "io_kind %d", io_kind);
    if (mode != SC_ATTN_STAGED && mode != SC_ATTN_FUSED) return sc_fail(SC_ERR_INVALID_ARG, "mode %d", mode);
    ScBatch b;
    st = make_batch(pool, n_seq, hist_lens, cu_new, max_blocks, sc_mma_tile_m(), &b);   // validate early
    if (st) return st;
    const bool staged = (mode == SC_ATTN_STAGED);
    if (staged && copy_stream == compute_stream)
        return sc_fail(SC_ERR_INVALID_ARG, "staged mode needs two different streams");
    cudaStream_t cs = (cudaStream_t)copy_stream, xs = (cudaStream_t)compute_stream;
    const ScGeom &g = pool->g;
    const int L = g.L, total_new = cu_new[n_seq];
    const int64_t q_bytes = (int64_t)total_new * g.Hq * g.D * 2, kv_bytes = (int64_t)total_new * g.Hkv * g.D * 2;
    const bool host_io = (io_kind == SC_MEM_HOST_PINNED);
    if (host_io && pool->stage_bytes == 0) {
        // Allocated ONCE, by the first host-I/O turn, for the largest turn the pool accepts (max_new_tokens):
        // q, out, k, v of one layer, two slots.  No later call allocates or frees (cudaMalloc / cudaFree
        // synchronise the device, and a turn that allocates cannot be captured into a graph).
        const int64_t mt = pool->cfg.max_new_tokens;
        const int64_t need = 2 * mt * g.Hq * g.D * 2 + 2 * mt * g.Hkv * g.D * 2;
        for (int i = 0; i < 2; ++i) {
            cudaError_t e = cudaMalloc((void **)&pool->stage[i], (size_t)need);
            if (e != cudaSuccess) {
                if (i == 1) { cudaFree(pool->stage[0]); pool->stage[0] = nullptr; }
                pool->stage[i] = nullptr;
                return sc_cuda_fail(e, "cudaMalloc(host-I/O staging)");
            }
        }
        pool->stage_bytes = need;
    }
    // fork: the side streams start after whatever the compute stream already holds
    SC_CUDA(cudaEventRecord(pool->ev_fork, xs));
    if (staged) {
        SC_CUDA(cudaStreamWaitEvent(cs, pool->ev_fork, 0));
        st = sc_load_layer_batched(pool, 0, tables_dev, max_blocks, n_seq, hist_lens, cu_new, 0, cs);
        if (st) return st;
        SC_CUDA(cudaEventRecord(pool->ev_load[0], cs));
    }
    if (host_io) {
        SC_CUDA(cudaStreamWaitEvent(pool->h2d_stream, pool->ev_fork, 0));
        SC_CUDA(cudaStreamWaitEvent(pool->d2h_stream, pool->ev_fork, 0));
    }
    for (int l = 0; l < L; ++l) {
        const int bf = (nbuf == 2) ? (l & 1) : 0;      // LSC buffer of this layer
        const int sb2 = l & 1;                         // host-io staging slot of this layer
        const char *q = (const char *)q_all + (int64_t)l * q_bytes;
        const char *k = (const char *)k_all + (int64_t)l * kv_bytes;
        const char *v = (const char *)v_all + (int64_t)l * kv_bytes;
        char *o = (char *)out_all + (int64_t)l * q_bytes;
        if (staged && nbuf == 2 && l + 1 < L) {
            // load(l+1) overwrites LSC[bf^1], last read by attention(l-1)
            if (l >= 1) SC_CUDA(cudaStreamWaitEvent(cs, pool->ev_attn[bf ^ 1], 0));
            st = sc_load_layer_batched(pool, l + 1, tables_dev, max_blocks, n_seq, hist_lens, cu_new, bf ^ 1, cs);
            if (st) return st;
            SC_CUDA(cudaEventRecord(pool->ev_load[bf ^ 1], cs));
        }
        const char *dq = q, *dk = k, *dv = v;
        char *dout = o;
        if (host_io) {
            char *sb = pool->stage[sb2];
            if (l >= 2) SC_CUDA(cudaStreamWaitEvent(pool->h2d_stream, pool->ev_comp[sb2], 0));
            SC_CUDA(cudaMemcpyAsync(sb, q, (size_t)q_bytes, cudaMemcpyHostToDevice, pool->h2d_stream));
            SC_CUDA(cudaMemcpyAsync(sb + q_bytes, k, (size_t)kv_bytes, cudaMemcpyHostToDevice, pool->h2d_stream));
            SC_CUDA(cudaMemcpyAsync(sb + q_bytes + kv_bytes, v, (size_t)kv_bytes, cudaMemcpyHostToDevice, pool->h2d_stream));
            SC_CUDA(cudaEventRecord(pool->ev_h2d[sb2], pool->h2d_stream));
            SC_CUDA(cudaStreamWaitEvent(xs, pool->ev_h2d[sb2], 0));
            if (l >= 2) SC_CUDA(cudaStreamWaitEvent(xs, pool->ev_d2h[sb2], 0));
            dq = sb; dk = sb + q_bytes; dv = sb + q_bytes + kv_bytes; dout = sb + q_bytes + 2 * kv_bytes;
        }
        if (staged) SC_CUDA(cudaStreamWaitEvent(xs, pool->ev_load[bf], 0));
        st = sc_prefill_layer_batched(pool, l, dq, dk, dv, tables_dev, max_blocks, n_seq, hist_lens, cu_new, bf,
                                      mode, dout, xs);
        if (st) return st;
        if (staged) SC_CUDA(cudaEventRecord(pool->ev_attn[bf], xs));
        if (staged && nbuf == 1 && l + 1 < L) {
            // the paper's ordering: load(l+1) into the ONE buffer waits for attention(l) and store(l)
            // (PAPER.md:192); it then runs beside whatever the hook puts on the compute stream
            SC_CUDA(cudaStreamWaitEvent(cs, pool->ev_attn[0], 0));
            st = sc_load_layer_batched(pool, l + 1, tables_dev, max_blocks, n_seq, hist_lens, cu_new, 0, cs);
            if (st) return st;
            SC_CUDA(cudaEventRecord(pool->ev_load[0], cs));
        }
        if (host_io) {
            SC_CUDA(cudaEventRecord(pool->ev_comp[sb2], xs));
            SC_CUDA(cudaStreamWaitEvent(pool->d2h_stream, pool->ev_comp[sb2], 0));
            SC_CUDA(cudaMemcpyAsync(o, dout, (size_t)q_bytes, cudaMemcpyDeviceToHost, pool->d2h_stream));
            SC_CUDA(cudaEventRecord(pool->ev_d2h[sb2], pool->d2h_stream));
        }
        if (opt && opt->after_attention) opt->after_attention(l, compute_stream, opt->user);
    }
    if (host_io) {   // join: the compute stream finishes last
        SC_CUDA(cudaStreamWaitEvent(xs, pool->ev_d2h[(L - 1) & 1], 0));
        if (L >= 2) SC_CUDA(cudaStreamWaitEvent(xs, pool->ev_d2h[(L - 2) & 1], 0));
    }
    return SC_OK;
}

sc_status_t sc_profile_enable(sc_pool_t *pool, int32_t on)
{
    if (!pool) return sc_fail(SC_ERR_INVALID_ARG, "pool is NULL");
    if (pool->host_only) return sc_fail(SC_ERR_CUDA, "host-only pool");
    for (auto &r : pool->prof) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    pool->prof.clear();
    pool->profiling = (on != 0);
    return SC_OK;
}

sc_status_t sc_profile_collect(sc_pool_t *pool, double *ms_sum, int64_t *count)
{
    if (!pool || !ms_sum || !count) return sc_fail(SC_ERR_INVALID_ARG, "NULL argument");
    for (int k = 0; k < SC_KERNEL_KINDS; ++k) { ms_sum[k] = 0; count[k] = 0; }
    for (auto &r : pool->prof) {
        SC_CUDA(cudaEventSynchronize(r.b));
        float ms = 0;
        SC_CUDA(cudaEventElapsedTime(&ms, r.a, r.b));
        ms_sum[r.kind] += ms;
        count[r.kind] += 1;
    }
    return SC_OK;
}

sc_status_t sc_launch_count(const sc_pool_t *pool, int64_t *n_launches)
{
    if (!pool || !n_launches) return sc_fail(SC_ERR_INVALID_ARG, "NULL argument");
    *n_launches = pool->launches;
    return SC_OK;
}

}  // extern "C"
