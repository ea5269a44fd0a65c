/*
 * oracle.c — TEST INFRASTRUCTURE, not the product.
 *
 * Plain, slow, single-threaded fp64 CPU statement of what the conserve_kv hot
 * path computes.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.
 * It shares no code, header, table or constant with paper_2606_01839_b200/ or
 * include/: the layout formulas below are typed out again from the prose of
 * DESIGN.md, on purpose.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md):
 *   - decode "generates each subsequent token by reading the full KV cache and
 *     appending one new entry"                     PAPER.md:50  §2.1
 *   - appends attend to "the whole history context" and compute KV "only ...
 *     for the appended tokens"                     PAPER.md:94  §3.1
 *   - the KV cache is "transferred once to the bound decoder"
 *                                                  PAPER.md:150 §4
 *   - provisioning Eq. 1, Eq. 2, R* = T_p / L_in   PAPER.md:162-172 §4.1
 *   - placement: lowest current KV occupancy       PAPER.md:176-178 §4.2
 * The paper writes no attention formula; it cites "Attention is all you need"
 * (PAPER.md:50).  The formula is therefore the textbook one,
 * softmax(q K^T / sqrt(d)) V, with the readings S1-S6 listed in DESIGN.md.
 *
 * Every function here is a definition written out, not the GPU's algorithm:
 * two-pass softmax (max, then sums), no online update, no partitioning, no
 * blocking.  Pins: tests/test_oracle_pins.py (closed forms, invariants, brute
 * force, torch float64 special cases).  Parity unpinned: none.
 *
 * Build: gcc -O2 -shared -fPIC -o liboracle.so oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* bf16 bit pattern -> double, exactly: bf16 is the top 16 bits of an fp32. */
static double bf16_to_double(uint16_t bits) {
    uint32_t u = ((uint32_t)bits) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* ------------------------------------------------------------------ O1 ----
 * Attention on LOGICAL (unpaged) KV.  One function serves decode and append.
 *   q [R][Hq][d], K [L][Hkv][d], V [L][Hkv][d]: bf16 bit patterns, logical
 *   token order.  R query rows are the LAST R positions: P = L - R, row i sits
 *   at position P + i and sees keys 0 .. P + i (n = P + i + 1 keys; decode is
 *   R = 1, n = L).  Query head h uses KV head h / G, G = Hq / Hkv.
 *   s_j = (sum_c q[i][h][c] K[j][g][c]) / sqrt(d)
 *   M = max_j s_j;  Z = sum_j exp(s_j - M);  LSE = M + ln Z
 *   O[i][h][c] = (sum_j exp(s_j - M) V[j][g][c]) / Z
 *   n = 0  ->  O = 0, LSE = -inf.
 * Outputs O [R][Hq][d] and LSE [R][Hq] as double.  Returns 0, or -1 on bad
 * arguments.  `scratch` holds L doubles (allocated here).
 */
int orc_attention(const uint16_t* q, const uint16_t* K, const uint16_t* V, int R, int L, int Hq, int Hkv,
                  int d, double* O, double* LSE) {
    /* R <= L (a row's own key is in the cache), except the one decode row on an EMPTY cache (R = 1, L = 0, so P = -1 and
     * n = 0): SURVEY 8c O1 step 6 / conserve_kv.h a4, O = 0 and LSE = -inf. */
    if (R < 0 || L < 0 || (R > L && !(R == 1 && L == 0)) || Hq <= 0 || Hkv <= 0 || d <= 0 || Hq % Hkv != 0) return -1;
    const int G = Hq / Hkv;
    const int P = L - R;
    const double inv_sqrt_d = 1.0 / sqrt((double)d);
    double* s = (double*)malloc(sizeof(double) * (size_t)(L > 0 ? L : 1));
    if (!s) return -1;
    for (int i = 0; i < R; ++i) {
        for (int h = 0; h < Hq; ++h) {
            const int g = h / G;
            const int n = P + i + 1;
            const uint16_t* qrow = q + ((size_t)i * Hq + h) * d;
            double* orow = O + ((size_t)i * Hq + h) * d;
            for (int c = 0; c < d; ++c) orow[c] = 0.0;
            if (n <= 0) {
                LSE[(size_t)i * Hq + h] = -INFINITY;
                continue;
            }
            double M = -INFINITY;
            for (int j = 0; j < n; ++j) {
                const uint16_t* krow = K + ((size_t)j * Hkv + g) * d;
                double acc = 0.0;
                for (int c = 0; c < d; ++c) acc += bf16_to_double(qrow[c]) * bf16_to_double(krow[c]);
                s[j] = acc * inv_sqrt_d;
                if (s[j] > M) M = s[j];
            }
            double Z = 0.0;
            for (int j = 0; j < n; ++j) {
                const double w = exp(s[j] - M);
                Z += w;
                const uint16_t* vrow = V + ((size_t)j * Hkv + g) * d;
                for (int c = 0; c < d; ++c) orow[c] += w * bf16_to_double(vrow[c]);
            }
            for (int c = 0; c < d; ++c) orow[c] /= Z;
            LSE[(size_t)i * Hq + h] = M + log(Z);
        }
    }
    free(s);
    return 0;
}

/* ----------------------------------------------------------- layout -------
 * Pool layout, restated from DESIGN.md ("Data layout in HBM"), in bf16 units.
 *   tile index  = ((layer * num_blocks + block) * 2 + kv) * Hkv + head
 *   tile size   = 16 * d
 *   in a tile, element (slot, c):
 *       half = c / 64, chunk = (c % 64) / 8, e = c % 8
 *       off  = half * 1024 + slot * 64 + ((chunk XOR (slot mod 8)) * 8) + e
 */
static size_t in_tile_offset(int slot, int c) {
    const int half = c / 64;
    const int chunk = (c % 64) / 8;
    const int e = c % 8;
    return (size_t)half * 1024u + (size_t)slot * 64u + (size_t)((chunk ^ (slot % 8)) * 8) + (size_t)e;
}

size_t orc_pool_addr(int num_blocks, int Hkv, int d, int layer, int block, int kv, int head, int slot, int c) {
    const size_t tile = (((size_t)layer * num_blocks + block) * 2u + (size_t)kv) * Hkv + head;
    return tile * (size_t)(16 * d) + in_tile_offset(slot, c);
}

size_t orc_pool_elems(int NL, int num_blocks, int Hkv, int d) {
    return (size_t)NL * num_blocks * 2u * Hkv * 16u * d;
}

/* ------------------------------------------------------------------ O2 ----
 * Reference gather, paged -> logical, one layer:
 *   K[t][g][c] = pool[addr(layer, table[t/16], 0, g, t%16, c)],  V with kv = 1.
 * Never reads table entries at or past ceil(L/16).
 */
int orc_gather(const uint16_t* pool, int num_blocks, int Hkv, int d, int layer, const int32_t* table, int L,
               uint16_t* K, uint16_t* V) {
    for (int t = 0; t < L; ++t) {
        const int block = table[t / 16];
        if (block < 0 || block >= num_blocks) return -1;
        for (int g = 0; g < Hkv; ++g)
            for (int c = 0; c < d; ++c) {
                K[((size_t)t * Hkv + g) * d + c] = pool[orc_pool_addr(num_blocks, Hkv, d, layer, block, 0, g, t % 16, c)];
                V[((size_t)t * Hkv + g) * d + c] = pool[orc_pool_addr(num_blocks, Hkv, d, layer, block, 1, g, t % 16, c)];
            }
    }
    return 0;
}

/* ------------------------------------------------------------------ O3 ----
 * Reference scatter = the handoff's result.  `pool` is the destination image
 * BEFORE the call (modified in place); k_src, v_src are [NL][tokens][Hkv][d].
 *   pool[addr(layer, table[(off+t)/16], kv, g, (off+t)%16, c)] = src_kv[layer][t][g][c]
 * as 16-bit assignments; nothing else is touched.
 */
int orc_scatter(uint16_t* pool, int NL, int num_blocks, int Hkv, int d, const uint16_t* k_src,
                const uint16_t* v_src, int tokens, int off, const int32_t* table, int n_ids) {
    if (tokens < 0 || off < 0) return -1;
    if (tokens > 0 && (off + tokens + 15) / 16 > n_ids) return -1;
    for (int layer = 0; layer < NL; ++layer)
        for (int t = 0; t < tokens; ++t) {
            const int pos = off + t;
            const int block = table[pos / 16];
            if (block < 0 || block >= num_blocks) return -1;
            for (int g = 0; g < Hkv; ++g)
                for (int c = 0; c < d; ++c) {
                    const size_t s = (((size_t)layer * tokens + t) * Hkv + g) * d + c;
                    pool[orc_pool_addr(num_blocks, Hkv, d, layer, block, 0, g, pos % 16, c)] = k_src[s];
                    pool[orc_pool_addr(num_blocks, Hkv, d, layer, block, 1, g, pos % 16, c)] = v_src[s];
                }
        }
    return 0;
}

/* Staging message, restated from DESIGN.md ("Staging message"):
 *   slot0 = off mod 16; ntb = ceil((slot0 + tokens) / 16);
 *   message = tiles [layer][tb][kv][head], each 16*d bf16 in the in-tile format;
 *   message token i is in tb = (slot0 + i) / 16, slot (slot0 + i) mod 16;
 *   slots carrying no token are zero.
 */
size_t orc_staging_elems(int NL, int Hkv, int d, int tokens, int off) {
    if (tokens <= 0) return 0;
    const int slot0 = off % 16;
    const int ntb = (slot0 + tokens + 15) / 16;
    return (size_t)NL * ntb * 2u * Hkv * 16u * d;
}

int orc_staging_message(int NL, int Hkv, int d, const uint16_t* k_src, const uint16_t* v_src, int tokens,
                        int off, uint16_t* msg) {
    if (tokens <= 0 || off < 0) return -1;
    const int slot0 = off % 16;
    const int ntb = (slot0 + tokens + 15) / 16;
    memset(msg, 0, sizeof(uint16_t) * orc_staging_elems(NL, Hkv, d, tokens, off));
    for (int layer = 0; layer < NL; ++layer)
        for (int i = 0; i < tokens; ++i) {
            const int tb = (slot0 + i) / 16, slot = (slot0 + i) % 16;
            for (int g = 0; g < Hkv; ++g)
                for (int c = 0; c < d; ++c) {
                    const size_t s = (((size_t)layer * tokens + i) * Hkv + g) * d + c;
                    const size_t tileK = (((size_t)layer * ntb + tb) * 2u + 0u) * Hkv + g;
                    const size_t tileV = (((size_t)layer * ntb + tb) * 2u + 1u) * Hkv + g;
                    msg[tileK * (size_t)(16 * d) + in_tile_offset(slot, c)] = k_src[s];
                    msg[tileV * (size_t)(16 * d) + in_tile_offset(slot, c)] = v_src[s];
                }
        }
    return 0;
}

/* ------------------------------------------------------------------ O4 ----
 * Merge identity (test helper): combine two normalised partial results over
 * disjoint key sets.  LSE = max + ln(exp(a - max) + exp(b - max)),
 * O = O_a exp(LSE_a - LSE) + O_b exp(LSE_b - LSE).  An empty side has
 * LSE = -inf and weight 0.
 */
void orc_merge(const double* Oa, double lse_a, const double* Ob, double lse_b, int d, double* O, double* lse) {
    if (lse_a == -INFINITY && lse_b == -INFINITY) {
        for (int c = 0; c < d; ++c) O[c] = 0.0;
        *lse = -INFINITY;
        return;
    }
    const double mx = lse_a > lse_b ? lse_a : lse_b;
    const double L = mx + log(exp(lse_a - mx) + exp(lse_b - mx));
    const double wa = (lse_a == -INFINITY) ? 0.0 : exp(lse_a - L);
    const double wb = (lse_b == -INFINITY) ? 0.0 : exp(lse_b - L);
    for (int c = 0; c < d; ++c) O[c] = Oa[c] * wa + Ob[c] * wb;
    *lse = L;
}

/* ---------------------------------------------------------- host rules ----
 * Provisioning, §4.1.  R* = T_p / L_in; Eq. 1: N T_d >= R L_d;
 * Eq. 2: N B >= R W; both at R = R*.  n_thr, n_mem are the real-valued lower
 * bounds; N the smallest integer meeting both.
 */
int orc_provision(double T_p, double L_in, double T_d, double L_d, double B, double W, double* rate,
                  double* n_thr, double* n_mem, int* N) {
    if (!(T_p > 0 && L_in > 0 && T_d > 0 && L_d > 0 && B > 0 && W > 0)) return -1;
    const double R = T_p / L_in;
    *rate = R;
    *n_thr = R * L_d / T_d;
    *n_mem = R * W / B;
    const double need = *n_thr > *n_mem ? *n_thr : *n_mem;
    *N = (int)ceil(need);
    return 0;
}

/* Placement, §4.2 ("lowest current KV cache occupancy") with the
 * readings S17: occupancy = used / total; ties -> lowest index; a decoder that
 * cannot hold `need` more blocks is skipped.  Returns the index
 * or -1 if none fits.
 */
int orc_place(const int* used, const int* total, int n, int need) {
    int best = -1;
    for (int i = 0; i < n; ++i) {
        if (total[i] - used[i] < need) continue;
        if (best < 0 || (long long)used[i] * total[best] < (long long)used[best] * total[i]) best = i;
    }
    return best;
}
