// sc_api.cu -- host side of libswiftcache.so: the C ABI of include/swiftcache.h.
// Pool descriptor, block allocator and block tables (a1, a2), argument checking,
// kernel dispatch (a3-a7, a9) and the layer-streaming pipeline (a8).
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "sc_internal.h"

static thread_local char g_err[512] = "";

sc_status_t sc_fail(sc_status_t code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof g_err, fmt, ap);
    va_end(ap);
    return code;
}

sc_status_t sc_cuda_fail(cudaError_t e, const char *what)
{
    return sc_fail(SC_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

const char *sc_err_buf() { return g_err; }

namespace {

#define SC_CUDA(call)                                                   \
    do {                                                                \
        cudaError_t e_ = (call);                                        \
        if (e_ != cudaSuccess) return sc_cuda_fail(e_, #call);             \
    } while (0)

inline int ceil_div(int a, int b) { return (a + b - 1) / b; }

sc_status_t make_geom(const sc_pool_config_t *c, ScGeom *g)
{
    if (!c) return sc_fail(SC_ERR_INVALID_ARG, "config is NULL");
    if (c->n_layers <= 0 || c->n_q_heads <= 0 || c->n_kv_heads <= 0 || c->n_blocks <= 0 ||
        c->lsc_blocks < 0 || c->max_new_tokens <= 0 || c->max_seqs <= 0)
        return sc_fail(SC_ERR_INVALID_ARG, "non-positive size in config");
    if (c->max_seqs > SC_MAX_SEQS) return sc_fail(SC_ERR_UNSUPPORTED, "max_seqs > %d", SC_MAX_SEQS);
    if (c->head_dim != 64 && c->head_dim != 128)
        return sc_fail(SC_ERR_UNSUPPORTED, "head_dim %d not in {64,128}", c->head_dim);
    if (c->block_size != 16) return sc_fail(SC_ERR_UNSUPPORTED, "block_size %d != 16", c->block_size);
    if (c->n_q_heads % c->n_kv_heads)
        return sc_fail(SC_ERR_UNSUPPORTED, "n_q_heads %d not a multiple of n_kv_heads %d", c->n_q_heads,
                    c->n_kv_heads);
    if (c->pool_kind != SC_POOL_HBM && c->pool_kind != SC_POOL_HOST_PINNED && c->pool_kind != SC_POOL_PEER)
        return sc_fail(SC_ERR_INVALID_ARG, "pool_kind %d", c->pool_kind);
    g->L = c->n_layers; g->Hq = c->n_q_heads; g->Hkv = c->n_kv_heads; g->D = c->head_dim;
    g->B = c->block_size; g->nh = c->head_dim / 64;
    g->chunk_bytes = (int64_t)g->B * g->D * 2;
    g->cell_bytes = 2 * (int64_t)g->Hkv * g->chunk_bytes;      // Eq. 1
    g->block_bytes = (int64_t)g->L * g->cell_bytes;            // block-major
    return SC_OK;
}

// splitmix64: seeds the free-list shuffle (S15: "shuffled pool" runs are reproducible)
inline uint64_t splitmix64(uint64_t &x)
{
    uint64_t z = (x += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

void destroy_resources(sc_pool *p)
{
    if (p->host_only) return;
    if (p->scratch) cudaFree(p->scratch);
    for (int i = 0; i < 2; ++i) {
        if (p->stage[i]) cudaFree(p->stage[i]);
        cudaEvent_t *evs[] = {&p->ev_load[i], &p->ev_attn[i], &p->ev_h2d[i], &p->ev_comp[i], &p->ev_d2h[i]};
        for (cudaEvent_t *e : evs)
            if (*e) cudaEventDestroy(*e);
    }
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->h2d_stream) cudaStreamDestroy(p->h2d_stream);
    if (p->d2h_stream) cudaStreamDestroy(p->d2h_stream);
}

}  // namespace

extern "C" {

const char *sc_version(void) { return "swiftcache-b200 0.1 (sm_100a)"; }
const char *sc_last_error(void) { return sc_err_buf(); }

sc_status_t sc_pool_bytes_required(const sc_pool_config_t *cfg, size_t *pool_bytes, size_t *lsc_bytes)
{
    ScGeom g;
    sc_status_t st = make_geom(cfg, &g);
    if (st) return st;
    if (!pool_bytes || !lsc_bytes) return sc_fail(SC_ERR_INVALID_ARG, "output pointer is NULL");
    *pool_bytes = (size_t)cfg->n_blocks * (size_t)g.block_bytes;
    *lsc_bytes = 2 * (size_t)cfg->lsc_blocks * (size_t)g.cell_bytes;
    return SC_OK;
}

sc_status_t sc_pool_create(const sc_pool_config_t *cfg, void *pool_base, size_t pool_bytes,
                           void *lsc_base, size_t lsc_bytes, int32_t zero_fill, sc_pool_t **out)
{
    ScGeom g;
    sc_status_t st = make_geom(cfg, &g);
    if (st) return st;
    if (!out) return sc_fail(SC_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    size_t need_pool, need_lsc;
    sc_pool_bytes_required(cfg, &need_pool, &need_lsc);
    const bool host_only = (pool_base == nullptr);
    if (!host_only) {
        if (pool_bytes < need_pool)
            return sc_fail(SC_ERR_CAPACITY, "pool region %zu < %zu bytes", pool_bytes, need_pool);
        if (((uintptr_t)pool_base & 1023) || ((uintptr_t)lsc_base & 1023))
            return sc_fail(SC_ERR_INVALID_ARG, "pool_base / lsc_base must be 1024-byte aligned");
        if (cfg->lsc_blocks > 0 && (!lsc_base || lsc_bytes < need_lsc))
            return sc_fail(SC_ERR_CAPACITY, "LSC region %zu < %zu bytes", lsc_bytes, need_lsc);
    }
    sc_pool *p = new (std::nothrow) sc_pool();
    if (!p) return sc_fail(SC_ERR_INVALID_ARG, "out of host memory");
    p->cfg = *cfg;
    p->g = g;
    p->pool_base = (char *)pool_base;
    p->lsc_base = (char *)lsc_base;
    p->pool_bytes = (int64_t)need_pool;
    p->lsc_buffer_bytes = (int64_t)cfg->lsc_blocks * g.cell_bytes;
    p->host_only = host_only;

    // free list: popped from the back, so store ids in reverse hand-out order
    p->free_list.resize(cfg->n_blocks);
    p->allocated.assign(cfg->n_blocks, 0);
    std::vector<int32_t> order(cfg->n_blocks);
    for (int i = 0; i < cfg->n_blocks; ++i) order[i] = i;
    if (cfg->alloc_seed) {
        uint64_t x = cfg->alloc_seed;
        for (int i = cfg->n_blocks - 1; i > 0; --i) {            // Fisher-Yates
            const int j = (int)(splitmix64(x) % (uint64_t)(i + 1));
            std::swap(order[i], order[j]);
        }
    }
    for (int i = 0; i < cfg->n_blocks; ++i) p->free_list[cfg->n_blocks - 1 - i] = order[i];

    if (!host_only) {
        int dev = 0, sms = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) { delete p; return sc_cuda_fail(e, "cudaGetDevice"); }
        p->n_sms = sms;
        p->max_splits = 32;
        const int64_t rows = (int64_t)cfg->max_new_tokens * g.Hq;
        const int64_t po = (int64_t)p->max_splits * rows * g.D * 4;
        const int64_t pml = (int64_t)p->max_splits * rows * 2 * 4;
        p->scratch_bytes = po + pml;
        e = cudaMalloc((void **)&p->scratch, (size_t)p->scratch_bytes);
        if (e != cudaSuccess) { delete p; return sc_cuda_fail(e, "cudaMalloc(scratch)"); }
        p->part_o = (float *)p->scratch;
        p->part_ml = (float *)(p->scratch + po);
        for (int i = 0; i < 2 && e == cudaSuccess; ++i) {
            cudaEvent_t *evs[] = {&p->ev_load[i], &p->ev_attn[i], &p->ev_h2d[i], &p->ev_comp[i], &p->ev_d2h[i]};
            for (cudaEvent_t *ev : evs)
                if (e == cudaSuccess) e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->h2d_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->d2h_stream, cudaStreamNonBlocking);
        if (e == cudaSuccess && zero_fill) {
            if (cfg->pool_kind == SC_POOL_HOST_PINNED) memset(pool_base, 0, need_pool);
            else e = cudaMemset(pool_base, 0, need_pool);
            if (e == cudaSuccess && lsc_base && need_lsc) e = cudaMemset(lsc_base, 0, need_lsc);
            if (e == cudaSuccess) e = cudaDeviceSynchronize();
        }
        if (e != cudaSuccess) {
            destroy_resources(p);
            delete p;
            return sc_cuda_fail(e, "sc_pool_create resources");
        }
    }
    *out = p;
    return SC_OK;
}

sc_status_t sc_pool_destroy(sc_pool_t *pool)
{
    if (!pool) return sc_fail(SC_ERR_INVALID_ARG, "pool is NULL");
    destroy_resources(pool);
    delete pool;
    return SC_OK;
}

sc_status_t sc_pool_info(const sc_pool_t *pool, sc_pool_info_t *info)
{
    if (!pool || !info) return sc_fail(SC_ERR_INVALID_ARG, "NULL argument");
    info->chunk_bytes = pool->g.chunk_bytes;
    info->cell_bytes = pool->g.cell_bytes;
    info->block_bytes = pool->g.block_bytes;
    info->pool_bytes = pool->pool_bytes;
    info->lsc_buffer_bytes = pool->lsc_buffer_bytes;
    info->lsc_bytes = 2 * pool->lsc_buffer_bytes;
    info->scratch_bytes = pool->scratch_bytes;
    {
        std::lock_guard<std::mutex> lk(const_cast<sc_pool_t *>(pool)->mu);     // the allocator calls are serialised
        info->n_free_blocks = (int32_t)pool->free_list.size();
    }
    info->max_splits = pool->max_splits;
    return SC_OK;
}

sc_status_t sc_cell_offset(const sc_pool_t *pool, int32_t block, int32_t layer, int32_t kv,
                           int32_t head, int32_t slot, int32_t d, int64_t *offset)
{
    if (!pool || !offset) return sc_fail(SC_ERR_INVALID_ARG, "NULL argument");
    const ScGeom &g = pool->g;
    if (block < 0 || block >= pool->cfg.n_blocks) return sc_fail(SC_ERR_BAD_BLOCK_ID, "block %d", block);
    if (layer < 0 || layer >= g.L || kv < 0 || kv > 1 || head < 0 || head >= g.Hkv || slot < 0 ||
        slot >= g.B || d < 0 || d >= g.D)
        return sc_fail(SC_ERR_INVALID_ARG, "coordinate out of range");
    *offset = (int64_t)block * g.block_bytes + (int64_t)layer * g.cell_bytes +
              (int64_t)(kv * g.Hkv + head) * g.chunk_bytes + sc_chunk_off(slot, d, g.nh);
    return SC_OK;
}

sc_status_t sc_lsc_offset(const sc_pool_t *pool, int32_t buf, int32_t lblock, int32_t kv,
                          int32_t head, int32_t slot, int32_t d, int64_t *offset)
{
    if (!pool || !offset) return sc_fail(SC_ERR_INVALID_ARG, "NULL argument");
    const ScGeom &g = pool->g;
    if (buf < 0 || buf > 1 || lblock < 0 || lblock >= pool->cfg.lsc_blocks || kv < 0 || kv > 1 ||
        head < 0 || head >= g.Hkv || slot < 0 || slot >= g.B || d < 0 || d >= g.D)
        return sc_fail(SC_ERR_INVALID_ARG, "coordinate out of range");
    *offset = (int64_t)buf * pool->lsc_buffer_bytes + (int64_t)lblock * g.cell_bytes +
              (int64_t)(kv * g.Hkv + head) * g.chunk_bytes + sc_chunk_off(slot, d, g.nh);
    return SC_OK;
}

sc_status_t sc_set_engine(sc_pool_t *pool, int32_t attn_engine, int32_t copy_engine)
{
    if (!pool) return sc_fail(SC_ERR_INVALID_ARG, "pool is NULL");
    if (attn_engine < SC_ENGINE_AUTO || attn_engine > SC_ENGINE_DECODE || copy_engine < SC_COPY_AUTO ||
        copy_engine > SC_COPY_BULK)
        return sc_fail(SC_ERR_INVALID_ARG, "unknown engine");
    pool->attn_engine = attn_engine;
    pool->copy_engine = copy_engine;
    return SC_OK;
}

sc_status_t sc_set_split_tiles(sc_pool_t *pool, int32_t tiles_per_split)
{
    if (!pool || tiles_per_split < 0) return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    pool->split_tiles_override = tiles_per_split;
    return SC_OK;
}

// --------------------------------------------------------------- a1 / a2
sc_status_t sc_alloc_blocks(sc_pool_t *pool, int32_t n, int32_t *ids_out)
{
    if (!pool || n < 0 || (n > 0 && !ids_out)) return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    std::lock_guard<std::mutex> lk(pool->mu);
    if ((size_t)n > pool->free_list.size())
        return sc_fail(SC_ERR_OUT_OF_BLOCKS, "need %d blocks, %zu free", n, pool->free_list.size());
    for (int i = 0; i < n; ++i) {
        const int32_t id = pool->free_list.back();
        pool->free_list.pop_back();
        pool->allocated[id] = 1;
        ids_out[i] = id;
    }
    return SC_OK;
}

sc_status_t sc_free_blocks(sc_pool_t *pool, const int32_t *ids, int32_t n)
{
    if (!pool || n < 0 || (n > 0 && !ids)) return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    std::lock_guard<std::mutex> lk(pool->mu);
    for (int i = 0; i < n; ++i) {               // validate first: all-or-nothing
        const int32_t id = ids[i];
        if (id < 0 || id >= pool->cfg.n_blocks || pool->allocated[id] != 1) {
            for (int j = 0; j < i; ++j) pool->allocated[ids[j]] = 1;
            return sc_fail(SC_ERR_BAD_BLOCK_ID, "block id %d is out of range, free, or repeated", id);
        }
        pool->allocated[id] = 2;                // mark: seen in this call
    }
    for (int i = 0; i < n; ++i) {
        pool->allocated[ids[i]] = 0;
        pool->free_list.push_back(ids[i]);
    }
    return SC_OK;
}

sc_status_t sc_num_free_blocks(const sc_pool_t *pool, int32_t *n_free)
{
    if (!pool || !n_free) return sc_fail(SC_ERR_INVALID_ARG, "NULL argument");
    std::lock_guard<std::mutex> lk(const_cast<sc_pool_t *>(pool)->mu);
    *n_free = (int32_t)pool->free_list.size();
    return SC_OK;
}

sc_status_t sc_append_blocks(sc_pool_t *pool, int32_t *table, int32_t *n_table, int32_t cap,
                             int32_t hist_len, int32_t n_new)
{
    if (!pool || !table || !n_table || hist_len < 0 || n_new < 0 || cap < 0 || *n_table < 0 ||
        *n_table > cap)
        return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    const int B = pool->g.B;
    if (*n_table < ceil_div(hist_len, B))
        return sc_fail(SC_ERR_INVALID_ARG, "table has %d entries but hist_len %d needs %d", *n_table,
                    hist_len, ceil_div(hist_len, B));
    const int64_t need = ((int64_t)hist_len + n_new + B - 1) / B;
    const int64_t add = need - *n_table;
    if (add <= 0) return SC_OK;
    if (need > cap) return sc_fail(SC_ERR_CAPACITY, "table capacity %d < %lld entries", cap, (long long)need);
    sc_status_t st = sc_alloc_blocks(pool, (int32_t)add, table + *n_table);
    if (st) return st;
    *n_table = (int32_t)need;
    return SC_OK;
}

// ---------------------------------------------- sizing and elasticity (f3, f1): host only
namespace {

// a * b for non-negative int64, false on overflow
bool mul_ok(int64_t a, int64_t b, int64_t *r) { return !__builtin_mul_overflow(a, b, r); }

sc_status_t block_elems_of(const sc_pool_config_t *c, int64_t *be)   // Eq. 6 / 7
{
    if (!c || c->n_layers <= 0 || c->block_size <= 0 || c->n_kv_heads <= 0 || c->head_dim <= 0)
        return sc_fail(SC_ERR_INVALID_ARG, "config needs positive n_layers, block_size, n_kv_heads, head_dim");
    int64_t v = c->n_layers;
    if (!mul_ok(v, c->block_size, &v) || !mul_ok(v, c->n_kv_heads, &v) || !mul_ok(v, c->head_dim, &v))
        return sc_fail(SC_ERR_CAPACITY, "block element count overflows int64");
    *be = v;
    return SC_OK;
}

}  // namespace

sc_status_t sc_lsc_rc_sizing(const sc_pool_config_t *cfg, int64_t c_master_bytes,
                             const int64_t *c_worker_bytes, int32_t n_workers, sc_sizing_t *out)
{
    if (!cfg || !out || n_workers < 0 || (n_workers > 0 && !c_worker_bytes) || c_master_bytes < 0)
        return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    if (cfg->n_layers <= 0 || cfg->block_size <= 0 || cfg->n_kv_heads <= 0 || cfg->head_dim <= 0)
        return sc_fail(SC_ERR_INVALID_ARG, "config needs positive n_layers, block_size, n_kv_heads, head_dim");
    // Eq. 1: one (block, layer) cell, K and V, bf16
    const int64_t m_block = 2ll * cfg->block_size * cfg->n_kv_heads * cfg->head_dim * 2;
    const int64_t full_layer_block = m_block * cfg->n_layers;
    sc_sizing_t r;
    r.k_master = c_master_bytes / m_block;                                   // Eq. 3
    r.sum_k = 0;
    for (int i = 0; i < n_workers; ++i) {
        if (c_worker_bytes[i] < 0) return sc_fail(SC_ERR_INVALID_ARG, "worker %d: negative size", i);
        r.sum_k += c_worker_bytes[i] / full_layer_block;                     // Eq. 2
    }
    const bool surplus = r.sum_k < r.k_master;
    r.n_lsc = surplus ? r.sum_k : r.k_master;                                // Eq. 4
    r.n_rc = surplus ? (r.k_master - r.sum_k) / cfg->n_layers : 0;           // Eq. 5
    r.max_context_blocks = r.n_lsc + r.n_rc;
    r.conventional_blocks = r.k_master / cfg->n_layers;
    *out = r;
    return SC_OK;
}

sc_status_t sc_elastic_units(const sc_pool_config_t *master, const sc_pool_config_t *worker,
                             int64_t *meu_master, int64_t *meu_worker)
{
    if (!meu_master || !meu_worker) return sc_fail(SC_ERR_INVALID_ARG, "output pointer is NULL");
    int64_t be_m, be_w;
    sc_status_t st = block_elems_of(master, &be_m);
    if (st) return st;
    st = block_elems_of(worker, &be_w);
    if (st) return st;
    int64_t x = be_m, y = be_w;                       // Euclid
    while (y != 0) { const int64_t t = x % y; x = y; y = t; }
    // LCM/BE_m = BE_w/gcd and LCM/BE_w = BE_m/gcd (Eq. 8-9) -- no need to form the LCM itself
    *meu_master = be_w / x;
    *meu_worker = be_m / x;
    return SC_OK;
}

sc_status_t sc_scale_up(int64_t n_worker_blocks, int32_t block_size, int64_t meu_worker,
                        int64_t meu_master, int64_t request_len, int64_t *d_worker, int64_t *d_master)
{
    if (!d_worker || !d_master || n_worker_blocks < 0 || block_size <= 0 || meu_worker <= 0 || meu_master <= 0 ||
        request_len < 0)
        return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    *d_worker = *d_master = 0;
    const int64_t need = request_len / block_size + (request_len % block_size != 0);
    if (need <= n_worker_blocks) return SC_OK;                                // enough capacity already
    const int64_t missing = need - n_worker_blocks;
    const int64_t units = missing / meu_worker + (missing % meu_worker != 0);  // whole elastic units, rounded up
    if (!mul_ok(units, meu_worker, d_worker) || !mul_ok(units, meu_master, d_master))
        return sc_fail(SC_ERR_CAPACITY, "block count overflows int64");
    return SC_OK;
}

sc_status_t sc_scale_down(int64_t n_worker_blocks, int32_t block_size, int64_t meu_worker,
                          int64_t meu_master, int64_t max_len, int64_t *d_worker, int64_t *d_master)
{
    if (!d_worker || !d_master || n_worker_blocks < 0 || block_size <= 0 || meu_worker <= 0 || meu_master <= 0 ||
        max_len < 0)
        return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    *d_worker = *d_master = 0;
    const int64_t max_need = max_len / block_size + (max_len % block_size != 0);
    if (max_need >= n_worker_blocks) return SC_OK;                            // the allocation is still needed
    const int64_t units = (n_worker_blocks - max_need) / meu_worker;          // whole elastic units, rounded down
    if (!mul_ok(units, meu_worker, d_worker) || !mul_ok(units, meu_master, d_master))
        return sc_fail(SC_ERR_CAPACITY, "block count overflows int64");
    return SC_OK;
}

sc_status_t sc_set_resident_blocks(sc_pool_t *pool, int32_t n_blocks)
{
    if (!pool || n_blocks < 0) return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    pool->resident_blocks = n_blocks;
    return SC_OK;
}

sc_status_t sc_pool_resize(sc_pool_t *pool, int32_t new_n_blocks, size_t new_pool_bytes,
                           int32_t zero_fill, void *stream)
{
    if (!pool || new_n_blocks <= 0) return sc_fail(SC_ERR_INVALID_ARG, "bad argument");
    std::lock_guard<std::mutex> lk(pool->mu);
    const int32_t old_n = pool->cfg.n_blocks;
    const size_t need = (size_t)new_n_blocks * (size_t)pool->g.block_bytes;
    if (new_n_blocks == old_n) return SC_OK;
    if (new_n_blocks > old_n) {
        if (!pool->host_only && new_pool_bytes < need)
            return sc_fail(SC_ERR_CAPACITY, "pool region %zu < %zu bytes", new_pool_bytes, need);
        if (!pool->host_only && zero_fill) {
            char *tail = pool->pool_base + (size_t)old_n * (size_t)pool->g.block_bytes;
            const size_t bytes = need - (size_t)old_n * (size_t)pool->g.block_bytes;
            if (pool->cfg.pool_kind == SC_POOL_HOST_PINNED) memset(tail, 0, bytes);
            else SC_CUDA(cudaMemsetAsync(tail, 0, bytes, (cudaStream_t)stream));
        }
        // Block-major: the new blocks are simply the next ids.  They go to the FRONT
        // of the free list (handed out last), so the tail stays free for a later shrink (S17).
        std::vector<int32_t> fresh;
        for (int32_t id = new_n_blocks - 1; id >= old_n; --id) fresh.push_back(id);
        pool->free_list.insert(pool->free_list.begin(), fresh.begin(), fresh.end());
        pool->allocated.resize(new_n_blocks, 0);
    } else {
        for (int32_t id = new_n_blocks; id < old_n; ++id)
            if (pool->allocated[id])
                return sc_fail(SC_ERR_BAD_BLOCK_ID, "cannot shrink to %d blocks: block %d is in use", new_n_blocks, id);
        pool->free_list.erase(std::remove_if(pool->free_list.begin(), pool->free_list.end(),
                                             [&](int32_t id) { return id >= new_n_blocks; }),
                              pool->free_list.end());
        pool->allocated.resize(new_n_blocks);
    }
    pool->cfg.n_blocks = new_n_blocks;
    pool->pool_bytes = (int64_t)need;
    return SC_OK;
}

}  // extern "C"
