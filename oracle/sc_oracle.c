/*
 * sc_oracle.c -- CPU oracle for the SwiftCache multi-turn prefill hot path.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call
 * this file.  It shares no code, header, table or helper with the CUDA path
 * under paper_2606_16135_b200/ and neither side includes the other.
 *
 * It is the plain definition of what the path computes, written slowly:
 *
 *   O1  pool model      block-major pool of NB full-layer blocks
 *                       (Sec. 3.4 "block-major layout",
 *                        PAPER.md:152 Eq. 1  M_block = 2*B*Hkv*Dkv*dtype)
 *   O2  store           token t of a conversation -> pool block table[t/B],
 *                       slot t%B (Sec. 3.3 "KV Store")
 *   O3  gather          pool -> contiguous per-layer history (the LSC content)
 *                       (Sec. 3.2 "preloads the KV cache for a
 *                        given layer into the LSC")
 *   O4  attention       each new token attends to every token that precedes
 *                       it, history plus new tokens up to and including
 *                       itself (Sec. 2.2, Fig. 2);
 *                       softmax scale 1/sqrt(D) (reading S1 in DESIGN.md)
 *   O5  append count    ceil((T_h+n)/B) - ceil(T_h/B) new table entries
 *                       (PAPER.md:142 block table; reading S10)
 *   O7  sizing          K_i, K_master, N_LSC, N_RC (Eq. 2-5); MEU / LCM
 *                       (Eq. 6-9); ScaleUp / ScaleDown (Algorithm 1)
 *
 * Precision: the north star fixes the oracle at fp32 ("a plain, slow CPU
 * fp32 implementation"); sco_attention_f64 is the same algorithm in double,
 * used by the tests to bound the fp32 oracle's own rounding error.
 * bf16 values travel as raw uint16_t bit patterns; copies are bit copies.
 *
 * Pins (tests/test_oracle_*.py, all "-m not gpu"): I1/I2 bit equality with
 * the logically contiguous tensor, I3 last-rows-of-monolithic-causal, I4
 * softmax row sums / V==1 / uniform closed form, I5 physical-permutation
 * invariance, I6 pure-Python float64 triple loop + torch SDPA on tiny,
 * Table 2 per-token KV bytes.  Nothing here is unpinned.
 *
 * OpenMP (if compiled with -fopenmp) only distributes independent
 * (query row, head) pairs over threads; the arithmetic per pair and its
 * order are unchanged.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ O1 -- */
/* The oracle's own internal order is [NB][L][2][B][Hkv][D]; parity is
 * defined on the logical accessor (p, l, kv, s, h, d), never on raw bytes. */
typedef struct {
    int32_t L, Hkv, D, B, NB;
    uint16_t *data; /* zero-initialised */
} sco_pool;

static size_t sco_index(const sco_pool *P, int p, int l, int kv, int s, int h, int d)
{
    size_t i = (size_t)p;
    i = i * (size_t)P->L + (size_t)l;
    i = i * 2u + (size_t)kv;
    i = i * (size_t)P->B + (size_t)s;
    i = i * (size_t)P->Hkv + (size_t)h;
    i = i * (size_t)P->D + (size_t)d;
    return i;
}

sco_pool *sco_pool_new(int32_t L, int32_t Hkv, int32_t D, int32_t B, int32_t NB)
{
    sco_pool *P = (sco_pool *)malloc(sizeof(sco_pool));
    if (!P) return NULL;
    P->L = L; P->Hkv = Hkv; P->D = D; P->B = B; P->NB = NB;
    size_t n = (size_t)NB * (size_t)L * 2u * (size_t)B * (size_t)Hkv * (size_t)D;
    P->data = (uint16_t *)calloc(n ? n : 1, sizeof(uint16_t));
    if (!P->data) { free(P); return NULL; }
    return P;
}

void sco_pool_free(sco_pool *P)
{
    if (P) { free(P->data); free(P); }
}

/* Eq. 1: bytes of one (block, layer) cell, K and V. */
int64_t sco_block_bytes(int32_t B, int32_t Hkv, int32_t D, int32_t dtype_bytes)
{
    return (int64_t)2 * B * Hkv * D * dtype_bytes;
}

/* Table 2: KV bytes per token over all layers. */
int64_t sco_kv_bytes_per_token(int32_t L, int32_t Hkv, int32_t D, int32_t dtype_bytes)
{
    return (int64_t)L * 2 * Hkv * D * dtype_bytes;
}

/* ------------------------------------------------------------------ O2 -- */
/* X is [n][Hkv][D] for ONE layer and ONE of K (kv=0) / V (kv=1); token i of
 * X is logical token start+i of the conversation whose table is `table`.
 * Returns 0, or -1 if a table entry is out of range.                       */
int sco_store(sco_pool *P, int32_t layer, int32_t kv, const uint16_t *X,
              int32_t start, int32_t n, const int32_t *table, int32_t n_table)
{
    for (int32_t i = 0; i < n; ++i) {
        int32_t t = start + i;
        int32_t lb = t / P->B, s = t % P->B;
        if (lb >= n_table) return -1;
        int32_t p = table[lb];
        if (p < 0 || p >= P->NB) return -1;
        for (int32_t h = 0; h < P->Hkv; ++h)
            for (int32_t d = 0; d < P->D; ++d)
                P->data[sco_index(P, p, layer, kv, s, h, d)] =
                    X[((size_t)i * P->Hkv + h) * P->D + d];
    }
    return 0;
}

/* ------------------------------------------------------------------ O3 -- */
/* out is [T][Hkv][D]: logical tokens 0..T-1 of one layer, K or V.          */
int sco_gather(const sco_pool *P, int32_t layer, int32_t kv, const int32_t *table,
               int32_t n_table, int32_t T, uint16_t *out)
{
    for (int32_t t = 0; t < T; ++t) {
        int32_t lb = t / P->B, s = t % P->B;
        if (lb >= n_table) return -1;
        int32_t p = table[lb];
        if (p < 0 || p >= P->NB) return -1;
        for (int32_t h = 0; h < P->Hkv; ++h)
            for (int32_t d = 0; d < P->D; ++d)
                out[((size_t)t * P->Hkv + h) * P->D + d] =
                    P->data[sco_index(P, p, layer, kv, s, h, d)];
    }
    return 0;
}

/* ------------------------------------------------------------------ O5 -- */
int32_t sco_blocks_for(int32_t tokens, int32_t B) { return (tokens + B - 1) / B; }

int32_t sco_append_count(int32_t hist_len, int32_t n_new, int32_t B)
{
    return sco_blocks_for(hist_len + n_new, B) - sco_blocks_for(hist_len, B);
}

/* ------------------------------------------------------------------ O4 -- */
static float sco_bf16_to_f32(uint16_t b)
{
    uint32_t u = (uint32_t)b << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return f;
}

/*
 * q    [n][Hq][D]      bf16 bits, the turn's new tokens
 * K, V [T_h+n][Hkv][D] bf16 bits, K = [history ; k_new], V likewise
 * out  [n][Hq][D]      REAL
 * rowsum (optional, may be NULL) [n][Hq]: sum_j p_j after normalisation
 *
 * For new token i, query head h, g = h / (Hq/Hkv):
 *   s_j = (sum_d q[i,h,d] * K[j,g,d]) / sqrt(D)      j = 0 .. T_h+i  (inclusive)
 *   m   = max_j s_j
 *   p_j = exp(s_j - m) / sum_j exp(s_j - m)
 *   out[i,h,:] = sum_j p_j * V[j,g,:]
 */
#define SCO_DEFINE_ATTENTION(NAME, REAL, EXPFN, SQRTFN)                               \
int NAME(const uint16_t *q, const uint16_t *K, const uint16_t *V, int32_t n,          \
         int32_t T_h, int32_t Hq, int32_t Hkv, int32_t D, REAL *out, REAL *rowsum)    \
{                                                                                     \
    if (n < 0 || T_h < 0 || Hq <= 0 || Hkv <= 0 || D <= 0 || Hq % Hkv) return -1;     \
    const int32_t G = Hq / Hkv;                                                       \
    const REAL scale = (REAL)1 / SQRTFN((REAL)D);                                     \
    int fail = 0;                                                                     \
    _Pragma("omp parallel for collapse(2) schedule(dynamic, 4)")                      \
    for (int32_t i = 0; i < n; ++i) {                                                 \
        for (int32_t h = 0; h < Hq; ++h) {                                            \
            const int32_t g = h / G;                                                  \
            const int32_t nk = T_h + i + 1;                                           \
            REAL *s = (REAL *)malloc((size_t)nk * sizeof(REAL));                      \
            if (!s) { fail = 1; continue; }                                           \
            const uint16_t *qi = q + ((size_t)i * Hq + h) * D;                        \
            REAL m = -INFINITY;                                                       \
            for (int32_t j = 0; j < nk; ++j) {                                        \
                const uint16_t *kj = K + ((size_t)j * Hkv + g) * D;                   \
                REAL acc = 0;                                                         \
                for (int32_t d = 0; d < D; ++d)                                       \
                    acc += (REAL)sco_bf16_to_f32(qi[d]) * (REAL)sco_bf16_to_f32(kj[d]); \
                s[j] = acc * scale;                                                   \
                if (s[j] > m) m = s[j];                                               \
            }                                                                         \
            REAL denom = 0;                                                           \
            for (int32_t j = 0; j < nk; ++j) { s[j] = EXPFN(s[j] - m); denom += s[j]; } \
            REAL psum = 0;                                                            \
            for (int32_t j = 0; j < nk; ++j) { s[j] = s[j] / denom; psum += s[j]; }   \
            REAL *o = out + ((size_t)i * Hq + h) * D;                                 \
            for (int32_t d = 0; d < D; ++d) o[d] = 0;                                 \
            for (int32_t j = 0; j < nk; ++j) {                                        \
                const uint16_t *vj = V + ((size_t)j * Hkv + g) * D;                   \
                for (int32_t d = 0; d < D; ++d)                                       \
                    o[d] += s[j] * (REAL)sco_bf16_to_f32(vj[d]);                      \
            }                                                                         \
            if (rowsum) rowsum[(size_t)i * Hq + h] = psum;                            \
            free(s);                                                                  \
        }                                                                             \
    }                                                                                 \
    return fail ? -2 : 0;                                                             \
}

SCO_DEFINE_ATTENTION(sco_attention_f32, float, expf, sqrtf)
SCO_DEFINE_ATTENTION(sco_attention_f64, double, exp, sqrt)

/* The softmax weights of one (query row, head), for tests of I4.
 * p_out has T_h+i+1 entries.                                               */
int sco_softmax_row_f32(const uint16_t *q, const uint16_t *K, int32_t T_h, int32_t i,
                        int32_t h, int32_t Hq, int32_t Hkv, int32_t D, float *p_out)
{
    if (Hq % Hkv) return -1;
    const int32_t g = h / (Hq / Hkv), nk = T_h + i + 1;
    const float scale = 1.0f / sqrtf((float)D);
    const uint16_t *qi = q + ((size_t)i * Hq + h) * D;
    float m = -INFINITY, denom = 0;
    for (int32_t j = 0; j < nk; ++j) {
        const uint16_t *kj = K + ((size_t)j * Hkv + g) * D;
        float acc = 0;
        for (int32_t d = 0; d < D; ++d) acc += sco_bf16_to_f32(qi[d]) * sco_bf16_to_f32(kj[d]);
        p_out[j] = acc * scale;
        if (p_out[j] > m) m = p_out[j];
    }
    for (int32_t j = 0; j < nk; ++j) { p_out[j] = expf(p_out[j] - m); denom += p_out[j]; }
    for (int32_t j = 0; j < nk; ++j) p_out[j] /= denom;
    return 0;
}

/* ---------------------------------------------------- sizing and elasticity -- */
/* Host integer arithmetic of Sec. 3.2 and 3.4-3.5, written out
 * as printed.  Pins: the worked example of PAPER.md:180 (tests/golden), lcm identities checked
 * against a brute-force search, hand-computed Algorithm 1 cases.                             */

/* Eq. 2-5 (the printed |.| of Eq. 2 and 5 are floors, reading S11).
 * c_master, c_worker[i]: KV cache bytes; m_block: Eq. 1; L: master layers.
 * out[0] = K_master (Eq. 3), out[1] = sum_i K_i (Eq. 2), out[2] = N_LSC (Eq. 4),
 * out[3] = N_RC (Eq. 5), out[4] = (N_LSC + N_RC) * 1 blocks = max context in blocks,
 * out[5] = floor(K_master / L): what a conventional full-layer cache holds.              */
int sco_lsc_rc_sizing(int64_t c_master, const int64_t *c_worker, int32_t n_workers,
                      int64_t m_block, int32_t L, int64_t *out)
{
    if (c_master < 0 || n_workers < 0 || m_block <= 0 || L <= 0) return -1;
    int64_t k_master = c_master / m_block;                       /* Eq. 3 */
    int64_t sum_k = 0;
    for (int32_t i = 0; i < n_workers; ++i) {
        if (c_worker[i] < 0) return -1;
        sum_k += c_worker[i] / (m_block * L);                    /* Eq. 2 */
    }
    int64_t n_lsc = sum_k < k_master ? sum_k : k_master;         /* Eq. 4 */
    int64_t n_rc = sum_k < k_master ? (k_master - sum_k) / L : 0;   /* Eq. 5 */
    out[0] = k_master; out[1] = sum_k; out[2] = n_lsc; out[3] = n_rc;
    out[4] = n_lsc + n_rc; out[5] = k_master / L;
    return 0;
}

/* Eq. 6-9: BE = L*B*Hkv*Dkv elements of one full-layer block;
 * LCM_elem = lcm(BE_m, BE_i); MEU_m = LCM/BE_m, MEU_i = LCM/BE_i.                        */
int64_t sco_block_elems(int32_t L, int32_t B, int32_t Hkv, int32_t D)
{
    return (int64_t)L * B * Hkv * D;
}

int sco_meu(int64_t be_m, int64_t be_i, int64_t *meu_m, int64_t *meu_i)
{
    if (be_m <= 0 || be_i <= 0) return -1;
    int64_t a = be_m, b = be_i;
    while (b) { int64_t t = a % b; a = b; b = t; }               /* a = gcd */
    int64_t lcm = be_m / a * be_i;                               /* Eq. 8 */
    *meu_m = lcm / be_m;                                         /* Eq. 9 */
    *meu_i = lcm / be_i;
    return 0;
}

/* Algorithm 1, ScaleUp: blocks the i-th worker gains and the master gives up. */
void sco_scale_up(int64_t n_i, int64_t b_i, int64_t meu_i, int64_t meu_m, int64_t request_len,
                  int64_t *d_worker, int64_t *d_master)
{
    int64_t need = (request_len + b_i - 1) / b_i;
    if (need <= n_i) { *d_worker = 0; *d_master = 0; return; }
    int64_t diff = need - n_i;
    int64_t k = (diff + meu_i - 1) / meu_i;
    *d_worker = k * meu_i; *d_master = k * meu_m;
}

/* Algorithm 1, ScaleDown: max_len = longest request of the last t seconds. */
void sco_scale_down(int64_t n_i, int64_t b_i, int64_t meu_i, int64_t meu_m, int64_t max_len,
                    int64_t *d_worker, int64_t *d_master)
{
    int64_t max_need = (max_len + b_i - 1) / b_i;
    if (max_need >= n_i) { *d_worker = 0; *d_master = 0; return; }
    int64_t diff = n_i - max_need;
    int64_t k = diff / meu_i;
    *d_worker = k * meu_i; *d_master = k * meu_m;
}

int sco_openmp_threads(void)
{
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    return omp_get_max_threads();
#else
    return 1;
#endif
}
