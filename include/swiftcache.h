/*
 * swiftcache.h -- C ABI of the B200-native SwiftCache multi-turn prefill hot path.
 *
 * What the library does (arxiv/paper_2606_16135, cited as PAPER.md:<line>):
 * for each transformer layer in turn, the conversation's historical KV is
 * fetched from a paged block pool through a block table into a small
 * active-layer buffer (the "layer stream cache", LSC, Sec. 3.2),
 * the turn's new tokens run causal attention over that history plus
 * themselves (Sec. 2.2), and their fresh K/V are scattered
 * back into pool blocks (Sec. 3.3).  Only the current
 * layer's KV, double-buffered, is resident in the LSC.
 *
 * Conventions
 *   - Plain C, no torch / C++ types.  Every pointer says HOST or DEVICE.
 *   - bf16 tensors are passed as `const void*` to raw bf16 bits.
 *   - Streams are passed as `void*` holding a cudaStream_t (0 = default stream).
 *   - Every call returns sc_status_t; SC_OK is 0.  sc_last_error() gives a
 *     thread-local message for the last failing call.  Argument errors are
 *     detected on the host before any launch; nothing is launched on error.
 *   - Data calls only ENQUEUE work on the given stream and return.  Ordering
 *     between different streams is the caller's job (or the pipeline
 *     helper's, sc_prefill_turn).
 *   - Threads: the allocator / table calls of one pool are serialised internally; the data
 *     calls of one pool (they share its scratch and counters) must come from one host
 *     thread at a time.  Different pools are independent.
 *   - Ownership: the sc_pool_t object and its internal scratch belong to the
 *     library.  pool_base / lsc_base and every tensor or table pointer are
 *     BORROWED from the caller and never freed here (the pool is *donated*
 *     memory in the paper too).
 *
 * Pool geometry ("block-major layout", Eq. 1)
 *   pool  = [n_blocks][n_layers] cells, each cell M_block = 2*B*Hkv*D*2 bytes
 *   cell  = [kv: K,V][Hkv] chunks, each chunk = the B=16 tokens x D values of
 *           one head, B*D*2 bytes, contiguous
 *   chunk = stored in the tensor core's 128-byte-swizzled operand order so a
 *           chunk is usable as a tcgen05.mma shared-memory operand after ONE
 *           contiguous bulk copy.  Byte offset of (slot s, dim d) in a chunk:
 *             (s/8)*(D/64)*1024 + (d/64)*1024 + (s%8)*128
 *               + ((((d%64)/8) ^ (s%8)) * 16) + (d%8)*2
 *           sc_cell_offset() returns the full byte offset; tests use it as
 *           the logical accessor.  The paper leaves the in-block order open
 *           (reading S3 in DESIGN.md).
 *   LSC   = 2 buffers x lsc_blocks cells in LOGICAL block order, same cell
 *           format, so a layer load is one contiguous M_block copy per block.
 */
#ifndef SWIFTCACHE_H_
#define SWIFTCACHE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sc_pool sc_pool_t; /* opaque, owned by the library */

typedef enum {
    SC_OK = 0,
    SC_ERR_INVALID_ARG = 1,   /* null pointer, negative size, layer out of range ...        */
    SC_ERR_OUT_OF_BLOCKS = 2, /* allocator exhausted; nothing was allocated                 */
    SC_ERR_CAPACITY = 3,      /* table / LSC / scratch too small for the request            */
    SC_ERR_BAD_BLOCK_ID = 4,  /* id out of range, double free, or not allocated             */
    SC_ERR_CUDA = 5,          /* a CUDA runtime call failed (also: no device present)       */
    SC_ERR_UNSUPPORTED = 6    /* head_dim not in {64,128}, block_size != 16, Hq % Hkv != 0  */
} sc_status_t;

/* where the pool region lives.  SC_POOL_PEER: the memory of ANOTHER GPU --
 * the paper's actual donor, "the worker GPU's idle memory ... accessed over NVLink" (PAPER.md:132,
 * :148, :332) -- mapped into this process by the caller (cudaDeviceEnablePeerAccess for a
 * same-process allocation, cudaIpcOpenMemHandle for another process's); every kernel addresses the
 * pool through pool_base only, so gather, scatter and fused attention read and write it across the
 * link exactly as they do local HBM.  The LSC is always local. */
typedef enum { SC_POOL_HBM = 0, SC_POOL_HOST_PINNED = 1, SC_POOL_PEER = 2 } sc_pool_kind_t;
typedef enum { SC_ATTN_STAGED = 0, SC_ATTN_FUSED = 1 } sc_attn_mode_t;
typedef enum { SC_MEM_DEVICE = 0, SC_MEM_HOST_PINNED = 1 } sc_mem_kind_t;
/* which attention engine sc_prefill_layer* uses; AUTO picks the fastest one
 * that supports the shape: SC_ENGINE_DECODE when every conversation of the call brings at most
 * 16 / (Hq / Hkv) new tokens (decode, n = 1: a paged read of the history, HBM-bound) and the call
 * reads at least 128 MiB of K/V per layer (below that the tcgen05 kernel's single launch per layer
 * wins), else SC_ENGINE_TCGEN05.  Forcing SC_ENGINE_DECODE on a call with more rows returns
 * SC_ERR_UNSUPPORTED. */
typedef enum { SC_ENGINE_AUTO = 0, SC_ENGINE_MMA_SYNC = 1, SC_ENGINE_TCGEN05 = 2, SC_ENGINE_DECODE = 3 } sc_engine_t;
/* which copy engine sc_load_layer* uses */
typedef enum { SC_COPY_AUTO = 0, SC_COPY_LDG = 1, SC_COPY_BULK = 2 } sc_copy_t;

typedef struct {
    int32_t n_layers;       /* L                                                          */
    int32_t n_q_heads;      /* Hq                                                         */
    int32_t n_kv_heads;     /* Hkv, must divide Hq                                        */
    int32_t head_dim;       /* D, 64 or 128                                               */
    int32_t block_size;     /* B tokens per block, must be 16                             */
    int32_t n_blocks;       /* pool capacity in full-layer blocks                         */
    int32_t pool_kind;      /* sc_pool_kind_t: where pool_base lives                      */
    int32_t lsc_blocks;     /* capacity of EACH of the two LSC buffers, in blocks         */
    int32_t max_new_tokens; /* most new tokens (summed over a batch) in one prefill call  */
    int32_t max_seqs;       /* most conversations in one batched call (>= 1)              */
    uint64_t alloc_seed;    /* 0: free list hands out ascending ids; else seeded shuffle  */
} sc_pool_config_t;

typedef struct {
    int64_t chunk_bytes;      /* B*D*2                                                    */
    int64_t cell_bytes;       /* M_block of Eq. 1 = 2*Hkv*chunk_bytes                     */
    int64_t block_bytes;      /* n_layers*cell_bytes: stride between pool blocks          */
    int64_t pool_bytes;       /* n_blocks*block_bytes                                     */
    int64_t lsc_buffer_bytes; /* lsc_blocks*cell_bytes: one of the two LSC buffers        */
    int64_t lsc_bytes;        /* 2*lsc_buffer_bytes                                       */
    int64_t scratch_bytes;    /* device scratch the library allocated for itself          */
    int32_t n_free_blocks;
    int32_t max_splits;       /* most split-KV partitions the attention may use           */
} sc_pool_info_t;

/* ------------------------------------------------------------------ lifecycle */

const char *sc_version(void);
/* Thread-local, static storage; valid until the next failing call on this thread. */
const char *sc_last_error(void);

/* Bytes the caller must provide for the pool region and for the LSC region (both
 * LSC buffers).  Pure host arithmetic (Eq. 1); works without a GPU.  HOST pointers. */
sc_status_t sc_pool_bytes_required(const sc_pool_config_t *cfg, size_t *pool_bytes, size_t *lsc_bytes);

/* pool_base: DEVICE pointer (SC_POOL_HBM), peer-DEVICE pointer valid on the current device
 * (SC_POOL_PEER) or pinned, device-mapped HOST pointer (SC_POOL_HOST_PINNED), 1024-byte aligned, >= pool_bytes.  lsc_base: DEVICE pointer,
 * 1024-byte aligned, >= lsc_bytes; may be NULL with lsc_blocks == 0 (fused mode only).
 * If zero_fill != 0 both regions are cleared; this is optional: the data path never
 * relies on what a slot it did not write holds (S10: the scatter of a turn zero-fills
 * the rest of the conversation's last block, every other unwritten slot is outside
 * what attention reads).  Passing pool_base == NULL creates a HOST-ONLY pool object: the
 * allocator / block-table calls work, every data call fails with SC_ERR_CUDA.       */
sc_status_t sc_pool_create(const sc_pool_config_t *cfg, void *pool_base, size_t pool_bytes,
                           void *lsc_base, size_t lsc_bytes, int32_t zero_fill, sc_pool_t **out);
sc_status_t sc_pool_destroy(sc_pool_t *pool);
sc_status_t sc_pool_info(const sc_pool_t *pool, sc_pool_info_t *info /* HOST */);

/* Logical accessor: byte offset from pool_base of element (block, layer, kv, head,
 * slot, d); kv = 0 for K, 1 for V.  *offset HOST.  Pure host arithmetic.            */
sc_status_t sc_cell_offset(const sc_pool_t *pool, int32_t block, int32_t layer, int32_t kv,
                           int32_t head, int32_t slot, int32_t d, int64_t *offset);
/* Same for the LSC: byte offset from lsc_base of (buf, logical block, kv, head, slot, d). */
sc_status_t sc_lsc_offset(const sc_pool_t *pool, int32_t buf, int32_t lblock, int32_t kv,
                          int32_t head, int32_t slot, int32_t d, int64_t *offset);

/* Select engines (defaults: AUTO).  Takes effect for later calls. */
sc_status_t sc_set_engine(sc_pool_t *pool, int32_t attn_engine /* sc_engine_t */,
                          int32_t copy_engine /* sc_copy_t */);
/* Force the number of split-KV tiles per partition (0 = automatic). */
sc_status_t sc_set_split_tiles(sc_pool_t *pool, int32_t tiles_per_split);

/* ------------------------------------------------- a1/a2: allocator and block tables
 * PAPER.md:142 (block table), :214-216 (block-major pool).  All arrays HOST.          */

/* All-or-nothing: on SC_ERR_OUT_OF_BLOCKS nothing is allocated.  Ids are distinct,
 * in [0, n_blocks), and were free (S15: which ids is unspecified).                    */
sc_status_t sc_alloc_blocks(sc_pool_t *pool, int32_t n, int32_t *ids_out);
/* SC_ERR_BAD_BLOCK_ID (and nothing freed) if any id is out of range, not allocated,
 * or repeated in the list.                                                            */
sc_status_t sc_free_blocks(sc_pool_t *pool, const int32_t *ids, int32_t n);
sc_status_t sc_num_free_blocks(const sc_pool_t *pool, int32_t *n_free);
/* Grow `table` (HOST array of capacity `cap`, currently *n_table entries) so that it
 * covers hist_len + n_new tokens: appends ceil((hist_len+n_new)/B) - *n_table fresh
 * ids (>= 0 of them).  Requires *n_table >= ceil(hist_len/B).  SC_ERR_CAPACITY if cap
 * is too small, SC_ERR_OUT_OF_BLOCKS if the pool is; in both cases nothing changes.   */
sc_status_t sc_append_blocks(sc_pool_t *pool, int32_t *table, int32_t *n_table, int32_t cap,
                             int32_t hist_len, int32_t n_new);

/* ------------------------------------------------------------------ data calls
 * Shapes use n = tokens, Hq/Hkv/D from the config.  "packed" means the sequences of
 * a batch are concatenated along the token axis.  SC_MAX_SEQS bounds a batch.       */
#define SC_MAX_SEQS 32

/* a3 -- PAPER.md:190 ("KV Store").  k, v: DEVICE bf16 [n_tokens][Hkv][D] of ONE layer,
 * written at logical tokens [start_token, start_token + n_tokens) of the conversation
 * whose table is table_dev (DEVICE int32[n_table], must cover the range).  Byte-exact. */
sc_status_t sc_store_prefix(sc_pool_t *pool, int32_t layer, const void *k, const void *v,
                            int32_t start_token, int32_t n_tokens, const int32_t *table_dev,
                            int32_t n_table, void *stream);

/* Inverse of a3, for verification and for callers that want contiguous KV back:
 * k_out, v_out DEVICE bf16 [n_tokens][Hkv][D] <- logical tokens [start, start+n).
 * src = 0: the pool through table_dev; src = 1 / 2: LSC buffer 0 / 1 (table_dev
 * ignored, logical block j is LSC block lsc_block_off + j).  Byte-exact.              */
sc_status_t sc_read_tokens(sc_pool_t *pool, int32_t layer, int32_t src, const int32_t *table_dev,
                           int32_t n_table, int32_t lsc_block_off, int32_t start_token,
                           int32_t n_tokens, void *k_out, void *v_out, void *stream);

/* a4 -- PAPER.md:148, :192 ("KV Load"): paged gather pool -> LSC[buf] of this layer's
 * first ceil(hist_len/B) blocks, in logical order (whole blocks are copied; S10).
 * SC_ERR_CAPACITY if they do not fit in lsc_blocks.  Enqueued on `stream` (the copy
 * stream).  The caller orders it before the sc_prefill_layer(STAGED) that reads buf
 * and after the previous reader of buf.                                               */
sc_status_t sc_load_layer(sc_pool_t *pool, int32_t layer, const int32_t *table_dev,
                          int32_t n_table, int32_t hist_len, int32_t buf, void *stream);

/* a5+a6+a7 -- PAPER.md:148, :190 (scatter), :72, :87 (attention).
 * q, out: DEVICE bf16 [n_new][Hq][D];  k_new, v_new: DEVICE bf16 [n_new][Hkv][D].
 * table_dev: DEVICE int32[n_table] covering hist_len + n_new tokens (sc_append_blocks).
 * Steps, all enqueued on `stream`:
 *   1. scatter k_new/v_new to logical tokens hist_len.. of the pool (and, in STAGED
 *      mode, to the same logical positions of LSC[buf]); the slots of the last block
 *      past token hist_len + n_new - 1 are set to zero;
 *   2. out[i,h,:] = sum_j softmax_j(q[i,h].K[j,h/G]/sqrt(D)) V[j,h/G,:], j <= hist_len+i,
 *      K/V = [history ; new], bf16 inputs, fp32 accumulation, bf16 output;
 *      STAGED reads LSC[buf] (history must have been loaded there), FUSED reads the
 *      pool blocks directly through table_dev and ignores buf;
 *   3. if the history was split across CTAs, the partial (m, l, O) triples are merged.
 * SC_ERR_CAPACITY: table too short, LSC too small (STAGED), n_new > max_new_tokens.
 * Append-only: step 1 treats hist_len + n_new as the END of the conversation.  Whatever the
 *   last block held behind token hist_len + n_new - 1 (up to 15 tokens) is overwritten with
 *   zeros, in the pool and in LSC[buf].  Re-running prefill over a middle slice of a
 *   conversation that is already stored further (recompute, evaluation) therefore destroys
 *   those tokens' K/V in that block; store them again (sc_store_prefix, which writes exactly
 *   the tokens it is given and pads nothing) or re-run the later turns.
 * table_dev (and tables_dev of the batched / turn calls) must be COMPLETE in device memory
 *   before the kernel that precedes this call on `stream` starts: the tcgen05 engine in FUSED
 *   mode is launched with programmatic dependent launch and reads the first table entries,
 *   through the read-only cache, while that preceding kernel may still be running.  A table
 *   written by a copy or kernel further back in the stream, or before a synchronisation, is
 *   fine (every use in this repository uploads the table once per turn); a table produced by
 *   the immediately preceding kernel is not.  q, k_new, v_new and the pool have no such
 *   restriction: they are read only after the preceding kernel's writes are visible.        */
sc_status_t sc_prefill_layer(sc_pool_t *pool, int32_t layer, const void *q, const void *k_new,
                             const void *v_new, const int32_t *table_dev, int32_t n_table,
                             int32_t hist_len, int32_t n_new, int32_t buf, int32_t mode,
                             void *out, void *stream);

/* a9 -- ragged batch (continuous batching is assumed by the paper).
 * tables_dev: DEVICE int32 [n_seq][max_blocks] (entries past a sequence's table are
 * ignored).  hist_lens, cu_new: HOST int32 [n_seq], [n_seq+1] (cu_new[0] = 0, new
 * tokens of sequence s are rows cu_new[s]..cu_new[s+1]-1 of the packed tensors).
 * In the LSC, sequence s starts at block sum_{t<s} ceil((hist_lens[t]+n_new[t])/B).    */
sc_status_t sc_load_layer_batched(sc_pool_t *pool, int32_t layer, const int32_t *tables_dev,
                                  int32_t max_blocks, int32_t n_seq, const int32_t *hist_lens,
                                  const int32_t *cu_new, int32_t buf, void *stream);
sc_status_t sc_prefill_layer_batched(sc_pool_t *pool, int32_t layer, const void *q,
                                     const void *k_new, const void *v_new,
                                     const int32_t *tables_dev, int32_t max_blocks, int32_t n_seq,
                                     const int32_t *hist_lens, const int32_t *cu_new, int32_t buf,
                                     int32_t mode, void *out, void *stream);

/* a8 -- the layer-streaming pipeline of one turn (ordering rule :192),
 * with the two-buffer reading S8 of DESIGN.md: for l = 0..L-1, the copy stream loads
 * layer l+1 into LSC[(l+1)%2] while the compute stream scatters + attends layer l from
 * LSC[l%2]; load(l+1) waits for attention(l-1), attention(l) waits for load(l).
 * Layers are issued strictly in order, one sc_prefill_layer_batched per layer.
 * q_all, out_all: [L][sum n_new][Hq][D]; k_all, v_all: [L][sum n_new][Hkv][D], bf16.
 * io_kind (sc_mem_kind_t): SC_MEM_DEVICE = DEVICE pointers; SC_MEM_HOST_PINNED = pinned
 * HOST pointers, in which case each layer's q/k/v are copied host->device and its out
 * device->host inside the call (double-buffered staging owned by the library: allocated ONCE,
 * by the first such call, for max_new_tokens -- 2 x max_new_tokens x (2 Hq + 2 Hkv) x D x 2
 * bytes; no later call allocates).
 * mode FUSED skips the loads.  On return all work is enqueued; compute_stream has been
 * made to wait for everything (synchronise it to wait for the turn).                   */
sc_status_t sc_prefill_turn(sc_pool_t *pool, const void *q_all, const void *k_all,
                            const void *v_all, void *out_all, int32_t io_kind,
                            const int32_t *tables_dev, int32_t max_blocks, int32_t n_seq,
                            const int32_t *hist_lens, const int32_t *cu_new, int32_t mode,
                            void *copy_stream, void *compute_stream);

/* a8 with options -- SURVEY.md 8(f) row f4.  The paper's own pipeline has ONE active-layer buffer
 * and hides the load behind the model's other work: "the (i)-th layer's load is blocked until
 * both the attention computation and KV store of the (i-1)-th layer are complete; the load then
 * overlaps with the FFN of layer i-1" (Fig. 10 at :404).
 *   lsc_buffers = 2 : sc_prefill_turn's schedule (reading S8): load(l+1) -> LSC[(l+1)%2] runs beside
 *                     attention(l) and waits for attention(l-1);
 *   lsc_buffers = 1 : the paper's: only LSC[0] is used; load(l+1) waits for attention(l) (which
 *                     follows the scatter = "KV store" of layer l on the same stream), attention(l+1)
 *                     waits for load(l+1).  Whatever the hook enqueues after attention(l) on the
 *                     compute stream (the model's o-proj / FFN) is what the load can hide behind.
 *   after_attention : may be NULL.  Called ON THE HOST, synchronously, once per layer, right after
 *                     layer l's attention (and, in STAGED mode with one buffer, the load of layer
 *                     l+1) has been enqueued; it may enqueue work on compute_stream and must not
 *                     synchronise.  The library neither reads nor writes what it enqueues.
 * opt == NULL means {2, NULL, NULL}.  Everything else as sc_prefill_turn.                       */
typedef void (*sc_layer_hook_t)(int32_t layer, void *compute_stream, void *user);
typedef struct {
    int32_t lsc_buffers;             /* 1 or 2 */
    sc_layer_hook_t after_attention; /* HOST callback, may be NULL */
    void *user;                      /* passed through to the hook */
} sc_turn_options_t;
sc_status_t sc_prefill_turn_ex(sc_pool_t *pool, const void *q_all, const void *k_all,
                               const void *v_all, void *out_all, int32_t io_kind,
                               const int32_t *tables_dev, int32_t max_blocks, int32_t n_seq,
                               const int32_t *hist_lens, const int32_t *cu_new, int32_t mode,
                               void *copy_stream, void *compute_stream, const sc_turn_options_t *opt);

/* a5+a6+a7 for callers that must not allocate -- same operation as sc_prefill_layer(FUSED):
 * scatter, attention over the pool blocks in place, merge
 * of the split-KV partitions.
 *
 * Why it exists.  Everything above needs an sc_pool_t, and sc_pool_create calls cudaMalloc (the
 * split-KV scratch) and creates streams and events.  Some callers cannot do that: a serving worker
 * that has already donated every spare byte of HBM to the block pool (PAPER.md:142, :148 -- there is
 * nothing left to allocate from, the call fails), and any caller on a live GPU that must not stall,
 * because cudaMalloc / cudaFree wait for the whole device and so hold up every stream on it.  This
 * call takes no pool object and allocates nothing, on the device or through any library: the partial
 * (m, l, O) results of the partitions go to a fixed array of SC_STATIC_SCRATCH_BYTES that is part of
 * the library's device image.  Every GPU on which the library's device code gets loaded holds that
 * array until the process exits, whether or not this call is ever made again.
 *
 * cfg: HOST; only n_layers, n_q_heads, n_kv_heads, head_dim and block_size are read (the geometry
 * of pool_base, exactly as in sc_pool_create).  pool_base: DEVICE (or peer / mapped pinned host)
 * pointer to the pool region, 1024-byte aligned; the caller owns it and guarantees it covers every
 * block id in table_dev.  q, out: DEVICE bf16 [n_new][Hq][D].  k_new, v_new: DEVICE bf16
 * [n_new][Hkv][D], stored at logical tokens hist_len.. first (rest of the last block zeroed, as
 * sc_prefill_layer does), or BOTH NULL if those tokens are in the pool already.  table_dev: DEVICE
 * int32[n_table] covering hist_len + n_new tokens.  Runs on the mma.sync engine.
 * tiles_per_split: 0 = the library picks the number of partitions and never picks more than fit in
 * the array; > 0 = that many 64-token KV tiles per partition (as sc_set_split_tiles; at most 32
 * partitions, longer ranges get larger partitions) -- for equal partitions the output is
 * bit-identical to sc_prefill_layer's.
 *
 * Limit: partitions x n_new x Hq x (D + 2) x 4 bytes (rounded up to 256) must not exceed
 * SC_STATIC_SCRATCH_BYTES, e.g. 7 partitions of 256 new tokens x 32 heads x D 128.  A forced split
 * beyond that returns SC_ERR_CAPACITY (message: bytes needed and the limit) and launches nothing;
 * one partition needs no scratch and always fits.  Other errors as sc_prefill_layer.
 *
 * First call on each GPU: looks up the array's device address (cudaGetSymbolAddress, with that GPU
 * current) and the SM count, and sets one kernel attribute; later calls only launch.  Make that
 * first call during start-up, outside any stream capture.
 * Sharing: there is ONE array per GPU for all callers and streams, and it keeps whatever the last
 * call wrote.  The call never depends on those old contents (every partial the merge reads is
 * written earlier in the same call, so nothing needs clearing), but two calls whose kernels can
 * overlap on one GPU -- different streams, different host threads -- race on it and both may
 * return garbage: issue them on one stream, or order them with events.  Enqueues up to three
 * kernels on `stream` and returns.                                                           */
#define SC_STATIC_SCRATCH_BYTES (32u << 20)
sc_status_t sc_prefill_layer_static(const sc_pool_config_t *cfg, void *pool_base, int32_t layer,
                                    const void *q, const void *k_new, const void *v_new,
                                    const int32_t *table_dev, int32_t n_table, int32_t hist_len,
                                    int32_t n_new, int32_t tiles_per_split, void *out, void *stream);

/* Per-kernel timing for measurement (bench.py's roofline): while enabled, every kernel
 * launch is bracketed by CUDA events on the stream it is launched on.  Enabling clears
 * earlier records.  sc_profile_collect waits for the recorded events and returns, per
 * kernel kind (sc_kernel_kind_t), the summed device time in ms and the launch count.
 * ms_sum, count: HOST arrays of SC_KERNEL_KINDS entries.                              */
typedef enum { SC_KERNEL_GATHER = 0, SC_KERNEL_SCATTER = 1, SC_KERNEL_ATTENTION = 2,
               SC_KERNEL_COMBINE = 3, SC_KERNEL_KINDS = 4 } sc_kernel_kind_t;
sc_status_t sc_profile_enable(sc_pool_t *pool, int32_t on);
sc_status_t sc_profile_collect(sc_pool_t *pool, double *ms_sum, int64_t *count);

/* Number of kernels the library has launched since the pool was created (all kinds). */
sc_status_t sc_launch_count(const sc_pool_t *pool, int64_t *n_launches);

/* ------------------------------------------- sizing and elasticity (host integer logic)
 * SURVEY.md 8(f) rows f3 and f1.  No device work, no data movement; all pointers HOST.   */

typedef struct {
    int64_t k_master;             /* Eq. 3: single-layer blocks the master's KV memory holds  */
    int64_t sum_k;                /* sum of Eq. 2 over the workers: full-layer blocks offered */
    int64_t n_lsc;                /* Eq. 4                                                    */
    int64_t n_rc;                 /* Eq. 5                                                    */
    int64_t max_context_blocks;   /* N_LSC + N_RC (x block_size = tokens)       */
    int64_t conventional_blocks;  /* floor(K_master / L): a cache without the LSC             */
} sc_sizing_t;

/* PAPER.md:150-180 (Sec. 3.2, Eq. 1-5).  cfg gives the master's L, Hkv, D, B (M_block, Eq. 1);
 * c_master_bytes / c_worker_bytes[i]: KV cache bytes of the master / the i-th worker.       */
sc_status_t sc_lsc_rc_sizing(const sc_pool_config_t *cfg, int64_t c_master_bytes,
                             const int64_t *c_worker_bytes, int32_t n_workers, sc_sizing_t *out);

/* PAPER.md:174-178 (regular cache, RC): the first n_blocks logical blocks of every conversation
 * are RESIDENT -- "stores KV cache directly on the master's local memory and retains full-layer
 * data ... requires no cross-GPU transfer".  In STAGED mode sc_load_layer* then skips them
 * (only later blocks are gathered into the LSC) and sc_prefill_layer* reads them in place
 * through the block table; FUSED mode is unaffected.  Only complete history blocks count
 * (min(n_blocks, hist_len / B) per conversation).  0 (default) = everything is streamed.
 * tcgen05 engine only (SC_ERR_UNSUPPORTED from a staged call with the mma.sync engine).      */
sc_status_t sc_set_resident_blocks(sc_pool_t *pool, int32_t n_blocks);

/* PAPER.md:218-304 (Sec. 3.4, Eq. 6-9): minimum elastic units.  Whenever the master moves
 * *meu_master of its full-layer blocks, the worker moves *meu_worker of its own, and both are
 * the same number of elements (their least common multiple).  Only n_layers, n_kv_heads,
 * head_dim and block_size of the two configs are read.  SC_ERR_CAPACITY on int64 overflow.  */
sc_status_t sc_elastic_units(const sc_pool_config_t *master, const sc_pool_config_t *worker,
                             int64_t *meu_master, int64_t *meu_worker);

/* PAPER.md:230-290 (Algorithm 1).  n_worker_blocks: blocks the worker holds now; block_size:
 * the worker's; request_len / max_len: tokens of the incoming request / of the longest request
 * of the last time window.  Outputs: blocks the worker gains (ScaleUp) or releases (ScaleDown)
 * and the blocks the master gives up or gains, both multiples of the elastic units.          */
sc_status_t sc_scale_up(int64_t n_worker_blocks, int32_t block_size, int64_t meu_worker,
                        int64_t meu_master, int64_t request_len, int64_t *d_worker, int64_t *d_master);
sc_status_t sc_scale_down(int64_t n_worker_blocks, int32_t block_size, int64_t meu_worker,
                          int64_t meu_master, int64_t max_len, int64_t *d_worker, int64_t *d_master);

/* PAPER.md:214-216 (block-major layout, Fig. 6): change the pool's capacity to new_n_blocks
 * full-layer blocks WITHOUT moving any block.  Growing appends block ids n_blocks ..
 * new_n_blocks-1 to the free list (the caller guarantees that the borrowed pool region
 * now extends to new_pool_bytes >= new_n_blocks * block_bytes from the same pool_base; the new
 * tail is zero-filled on `stream` if zero_fill != 0).  Shrinking releases the LAST blocks
 * and is refused with SC_ERR_BAD_BLOCK_ID, changing nothing, unless every one of them is free
 * (reading S17).  Offsets of surviving blocks (sc_cell_offset) do not change.               */
sc_status_t sc_pool_resize(sc_pool_t *pool, int32_t new_n_blocks, size_t new_pool_bytes,
                           int32_t zero_fill, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* SWIFTCACHE_H_ */
