/*
 * anslin ORACLE — TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct CPU restatement of the codec the paper describes
 * (arxiv/paper_2606_15789, /root/reference/PAPER.md = "P").  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with
 * paper_2606_15789_b200/csrc (the product); the only thing both sides read is the byte-level
 * container description in DESIGN.md.
 *
 * Every function follows the paper's order and notation, with (b, w, L) as run-time parameters so
 * that the hand-worked Examples A and B (tests/golden/) run through the very same code:
 *   b  = probability bits, M = 2^b slots           (P:l.440-442, Eq.3: "2^b" entries, default b=12)
 *   w  = bits per renormalisation word             (P:l.281-285, Alg V.2 l.9-11; reading A3: w=16)
 *   L  = lower bound of the normalised state interval [L, L*2^w)   (reading A3: L = 2^16)
 *
 * No blocking, fusion, tables-of-tables or reordering beyond what the algorithm states.
 * Pins (tests/test_oracle_*.py): worked Examples A and B, power-of-two closed form, uniform
 * table special case, brute-force unique decodability on tiny alphabets, final-state invariant,
 * scipy entropy, Gibbs inequality, Table III via Eq.3.
 */
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>

/* ---- P:l.68-72 (§II-B): empirical histogram and Shannon entropy H = -sum p_i log2 p_i ---- */
void orc_histogram(const uint8_t *sym, size_t n, uint64_t *cnt /*[256]*/)
{
    for (int s = 0; s < 256; ++s) cnt[s] = 0;
    for (size_t i = 0; i < n; ++i) cnt[sym[i]] += 1;
}

double orc_entropy(const uint64_t *cnt, int nsym)
{
    double n = 0.0, h = 0.0;
    for (int s = 0; s < nsym; ++s) n += (double)cnt[s];
    if (n == 0.0) return 0.0;
    for (int s = 0; s < nsym; ++s) {
        if (cnt[s] == 0) continue;
        double p = (double)cnt[s] / n;
        h -= p * log2(p);
    }
    return h;
}

/* Cross entropy of the data under the quantised table: sum p_s log2(M / f_s) */
double orc_cross_entropy(const uint64_t *cnt, const uint32_t *f, int nsym, int b)
{
    double n = 0.0, x = 0.0, M = (double)(1u << b);
    for (int s = 0; s < nsym; ++s) n += (double)cnt[s];
    if (n == 0.0) return 0.0;
    for (int s = 0; s < nsym; ++s) {
        if (cnt[s] == 0) continue;
        x += ((double)cnt[s] / n) * log2(M / (double)f[s]);
    }
    return x;
}

/*
 * Frequency normalisation to sum 2^b (P:l.366 "finite-precision normalization"; the paper is
 * silent on the method -> DESIGN.md reading A10): f_s >= 1 iff cnt_s > 0, sum f = M, greedy on
 * the separable objective sum cnt_s*log2(f_s); ties -> smallest symbol.  Degenerate histogram
 * with a single live symbol (reading A11): f = M-1 for it and 1 for symbol (s+1) mod nsym, so
 * that every f fits b bits.  Returns 0, or -1 if there are more live symbols than slots / none.
 */
int orc_normalize(const uint64_t *cnt, int nsym, int b, uint32_t *f)
{
    const uint32_t M = 1u << b;
    double n = 0.0;
    int live = 0, only = -1;
    for (int s = 0; s < nsym; ++s) { n += (double)cnt[s]; if (cnt[s]) { ++live; only = s; } }
    if (live == 0 || (uint32_t)live > M) return -1;
    if (live == 1) {
        for (int s = 0; s < nsym; ++s) f[s] = 0;
        f[only] = M - 1;
        f[(only + 1) % nsym] = 1;
        return 0;
    }
    uint64_t sum = 0;
    for (int s = 0; s < nsym; ++s) {
        if (cnt[s] == 0) { f[s] = 0; continue; }
        uint64_t q = (uint64_t)floor((double)cnt[s] * (double)M / n);
        f[s] = q < 1 ? 1u : (uint32_t)q;
        sum += f[s];
    }
    while (sum < M) {               /* give +1 where it buys the most bits */
        int best = -1; double gain = -1.0;
        for (int s = 0; s < nsym; ++s) {
            if (cnt[s] == 0) continue;
            double g = (double)cnt[s] * log2(((double)f[s] + 1.0) / (double)f[s]);
            if (g > gain) { gain = g; best = s; }
        }
        f[best] += 1; sum += 1;
    }
    while (sum > M) {               /* take 1 where it costs the fewest bits */
        int best = -1; double cost = 0.0;
        for (int s = 0; s < nsym; ++s) {
            if (cnt[s] == 0 || f[s] <= 1) continue;
            double c = (double)cnt[s] * log2((double)f[s] / ((double)f[s] - 1.0));
            if (best < 0 || c < cost) { cost = c; best = s; }
        }
        f[best] -= 1; sum -= 1;
    }
    return 0;
}

/* c_s = exclusive prefix sum of f in symbol order (P:l.271 table entry (sigma, f, c)) */
void orc_cumulative(const uint32_t *f, int nsym, uint32_t *c)
{
    uint32_t acc = 0;
    for (int s = 0; s < nsym; ++s) { c[s] = acc; acc += f[s]; }
}

/* slot -> symbol: the unique s with c_s <= slot < c_s + f_s (P:l.271, Alg V.2 l.5) */
void orc_slot_table(const uint32_t *f, const uint32_t *c, int nsym, int b, uint8_t *sym_of_slot)
{
    for (int s = 0; s < nsym; ++s)
        for (uint32_t k = 0; k < f[s]; ++k) sym_of_slot[c[s] + k] = (uint8_t)s;
    (void)b;
}

/*
 * Textbook rANS (Duda, ref [13] P:l.506), the encoder that Alg V.2 (P:l.260-287) inverts.
 * One encoding step of symbol s on state x.  Emitted words are appended to out[*n_out] in
 * EMISSION order.  (SURVEY 8(c) step 6.)
 */
static uint64_t enc_step(uint64_t x, uint32_t fs, uint32_t cs, int b, int w, int Llog2,
                         uint16_t *out, size_t *n_out)
{
    const uint64_t L = 1ull << Llog2;
    const uint64_t x_max = ((L >> b) << w) * (uint64_t)fs;
    const uint64_t wmask = (1ull << w) - 1;
    while (x >= x_max) {
        out[(*n_out)++] = (uint16_t)(x & wmask);
        x >>= w;
    }
    return ((x / fs) << b) + cs + (x % fs);
}

/*
 * Scalar encode of one stream sym[0..n-1].  Symbols are encoded last-to-first so that the decoder
 * produces them first-to-last.  words_dec receives the words in DECODER read order (reverse of
 * emission).  Returns the number of words; *state_out is the state the decoder starts from.
 */
size_t orc_encode_scalar(const uint8_t *sym, size_t n, const uint32_t *f, const uint32_t *c,
                         int b, int w, int Llog2, uint64_t x_init,
                         uint64_t *state_out, uint16_t *words_dec)
{
    size_t cap = n * 2 + 8, nw = 0;
    uint16_t *emit = (uint16_t *)malloc(cap * sizeof(uint16_t));
    uint64_t x = x_init;
    for (size_t i = n; i-- > 0;) x = enc_step(x, f[sym[i]], c[sym[i]], b, w, Llog2, emit, &nw);
    for (size_t k = 0; k < nw; ++k) words_dec[k] = emit[nw - 1 - k];
    free(emit);
    *state_out = x;
    return nw;
}

/*
 * Scalar decode, Alg V.2 l.3-11 (P:l.267-285) for one lane:
 *   slot = x mod M; (sigma,f,c) = T[slot]; out = sigma; x = f*floor(x/M) + (slot - c);
 *   while x < L: x = (x << w) | next word.
 * Returns the number of words consumed; *state_end is the state after the last symbol
 * (== the encoder's x_init: integrity invariant).
 */
size_t orc_decode_scalar(uint64_t state, const uint16_t *words, size_t n,
                         const uint32_t *f, const uint32_t *c, const uint8_t *sym_of_slot,
                         int b, int w, int Llog2, uint8_t *out, uint64_t *state_end)
{
    const uint64_t M = 1ull << b, L = 1ull << Llog2;
    uint64_t x = state;
    size_t r = 0;
    for (size_t i = 0; i < n; ++i) {
        uint64_t slot = x & (M - 1);
        uint8_t s = sym_of_slot[slot];
        out[i] = s;
        x = (uint64_t)f[s] * (x >> b) + (slot - c[s]);
        while (x < L) x = (x << w) | words[r++];
    }
    *state_end = x;
    return r;
}

/*
 * R-lane interleaved tile encode (P:l.192 "R independent substreams", l.256 "interleaved across
 * lanes ... renormalization loads are naturally coalesced").
 * Tile symbol i belongs to lane i mod R at step i div R.  The decoder's read order DEFINES the
 * layout: after decoding step t, the lanes that must renormalise read consecutive words in
 * ascending lane order.  The encoder obtains that order by running the schedule backwards
 * (t descending, lane descending) with ONE shared stack of emitted words.
 * n must be a multiple of R.  x_init[R] are the encoder start states (decoder end states).
 */
size_t orc_tile_encode(const uint8_t *sym, size_t n, int R, const uint32_t *f, const uint32_t *c,
                       int b, int w, int Llog2, const uint64_t *x_init,
                       uint64_t *states_out /*[R]*/, uint16_t *words_dec)
{
    size_t steps = n / (size_t)R, cap = n * 2 + 8, nw = 0;
    uint16_t *emit = (uint16_t *)malloc(cap * sizeof(uint16_t));
    uint64_t *x = (uint64_t *)malloc((size_t)R * sizeof(uint64_t));
    for (int l = 0; l < R; ++l) x[l] = x_init[l];
    for (size_t t = steps; t-- > 0;)
        for (int l = R; l-- > 0;) {
            uint8_t s = sym[t * (size_t)R + (size_t)l];
            x[l] = enc_step(x[l], f[s], c[s], b, w, Llog2, emit, &nw);
        }
    for (size_t k = 0; k < nw; ++k) words_dec[k] = emit[nw - 1 - k];
    for (int l = 0; l < R; ++l) states_out[l] = x[l];
    free(emit); free(x);
    return nw;
}

/* R-lane interleaved tile decode = Alg V.2 executed by R lanes in lock step. */
size_t orc_tile_decode(const uint64_t *states /*[R]*/, const uint16_t *words, size_t n, int R,
                       const uint32_t *f, const uint32_t *c, const uint8_t *sym_of_slot,
                       int b, int w, int Llog2, uint8_t *out, uint64_t *states_end /*[R]*/)
{
    const uint64_t M = 1ull << b, L = 1ull << Llog2;
    size_t steps = n / (size_t)R, r = 0;
    uint64_t *x = (uint64_t *)malloc((size_t)R * sizeof(uint64_t));
    for (int l = 0; l < R; ++l) x[l] = states[l];
    for (size_t t = 0; t < steps; ++t)
        for (int l = 0; l < R; ++l) {
            uint64_t slot = x[l] & (M - 1);
            uint8_t s = sym_of_slot[slot];
            out[t * (size_t)R + (size_t)l] = s;
            x[l] = (uint64_t)f[s] * (x[l] >> b) + (slot - c[s]);
            while (x[l] < L) x[l] = (x[l] << w) | words[r++];
        }
    for (int l = 0; l < R; ++l) states_end[l] = x[l];
    free(x);
    return r;
}

/*
 * Second, independent formulation of the interleave ("plain alternative"):
 * encode every lane on its own with the scalar encoder, then SIMULATE the lock-step decoder and
 * hand each request the next word of the requesting lane's private queue.  Must give the same
 * bytes as orc_tile_encode; tests use one to check the other.
 */
size_t orc_tile_encode_by_simulation(const uint8_t *sym, size_t n, int R, const uint32_t *f,
                                     const uint32_t *c, const uint8_t *sym_of_slot,
                                     int b, int w, int Llog2, const uint64_t *x_init,
                                     uint64_t *states_out, uint16_t *words_dec)
{
    const uint64_t M = 1ull << b, L = 1ull << Llog2;
    size_t steps = n / (size_t)R;
    uint8_t *lane_sym = (uint8_t *)malloc(steps ? steps : 1);
    uint16_t **q = (uint16_t **)malloc((size_t)R * sizeof(uint16_t *));
    size_t *qn = (size_t *)malloc((size_t)R * sizeof(size_t));
    size_t *qr = (size_t *)calloc((size_t)R, sizeof(size_t));
    uint64_t *x = (uint64_t *)malloc((size_t)R * sizeof(uint64_t));
    for (int l = 0; l < R; ++l) {
        for (size_t t = 0; t < steps; ++t) lane_sym[t] = sym[t * (size_t)R + (size_t)l];
        q[l] = (uint16_t *)malloc((steps * 2 + 8) * sizeof(uint16_t));
        qn[l] = orc_encode_scalar(lane_sym, steps, f, c, b, w, Llog2, x_init[l], &states_out[l], q[l]);
        x[l] = states_out[l];
    }
    size_t nw = 0;
    for (size_t t = 0; t < steps; ++t)
        for (int l = 0; l < R; ++l) {
            uint64_t slot = x[l] & (M - 1);
            uint8_t s = sym_of_slot[slot];
            x[l] = (uint64_t)f[s] * (x[l] >> b) + (slot - c[s]);
            while (x[l] < L) {
                uint16_t word = q[l][qr[l]++];
                words_dec[nw++] = word;
                x[l] = (x[l] << w) | word;
            }
        }
    for (int l = 0; l < R; ++l) free(q[l]);
    free(q); free(qn); free(qr); free(x); free(lane_sym);
    return nw;
}

/*
 * Lane stream with in-stream literals: a coded symbol holds two
 * 4-bit codes (low nibble = first weight); code 15 is an escape whose true value follows in the lane's own word
 * stream.  Steps come in chunks of four (eight weights = one 16-byte bf16 operand chunk): the decoder decodes and
 * renormalises the four steps (0 or 1 word each), then reads one literal word per escaped nibble of the chunk, in
 * weight order (step by step, low nibble first).  lit[] holds all literals consecutively in weight order.  n % 4 == 0.
 * words_dec receives the stream in decoder read order; after_step[i] = words consumed once step i is complete
 * (so a caller can cut the stream into segments of steps).  Returns the total number of words.
 */
size_t orc_encode_scalar_lit(const uint8_t *sym, size_t n, const uint32_t *f, const uint32_t *c,
                             int b, int w, int Llog2, uint64_t x_init, const uint16_t *lit,
                             uint64_t *state_out, uint16_t *words_dec, uint32_t *after_step)
{
    /* plain rANS first: emitted[i] = words the encoder put out BEFORE coding symbol i = what the decoder's
     * renormalisation after step i reads */
    uint16_t *emit = (uint16_t *)malloc((n * 2 + 8) * sizeof(uint16_t));
    uint32_t *first = (uint32_t *)malloc((n + 1) * sizeof(uint32_t));   /* emission index range of step i: [first[i+1].. first[i]) in emission order */
    size_t nw = 0;
    uint64_t x = x_init;
    for (size_t i = n; i-- > 0;) {
        first[i + 1] = (uint32_t)nw;   /* emissions so far belong to later steps */
        x = enc_step(x, f[sym[i]], c[sym[i]], b, w, Llog2, emit, &nw);
    }
    first[0] = (uint32_t)nw;
    /* emissions of step i (made while coding symbol i) occupy emission indices [first[i+1], first[i]) */
    size_t out = 0, li = 0;
    for (size_t i = 0; i < n; ++i) {
        for (uint32_t k = first[i]; k-- > first[i + 1];) words_dec[out++] = emit[k];   /* decoder reads them in reverse emission order */
        if ((i & 3) == 3)
            for (size_t j = i - 3; j <= i; ++j) {
                if ((sym[j] & 15) == 15) words_dec[out++] = lit[li++];
                if ((sym[j] >> 4) == 15) words_dec[out++] = lit[li++];
            }
        after_step[i] = (uint32_t)out;
    }
    free(emit); free(first);
    *state_out = x;
    return out;
}

/* Inverse of orc_encode_scalar_lit.  out_lit[2i], out_lit[2i+1]: the literal of step i's low / high nibble, or 0xFFFF
 * when that nibble is not an escape.  Returns the number of words consumed. */
size_t orc_decode_scalar_lit(uint64_t state, const uint16_t *words, size_t n,
                             const uint32_t *f, const uint32_t *c, const uint8_t *sym_of_slot,
                             int b, int w, int Llog2, uint8_t *out, uint16_t *out_lit, uint64_t *state_end)
{
    const uint64_t M = 1ull << b, L = 1ull << Llog2;
    uint64_t x = state;
    size_t r = 0;
    for (size_t i = 0; i < n; ++i) {
        uint64_t slot = x & (M - 1);
        uint8_t s = sym_of_slot[slot];
        out[i] = s;
        x = (uint64_t)f[s] * (x >> b) + (slot - c[s]);
        while (x < L) x = (x << w) | words[r++];
        if ((i & 3) == 3)
            for (size_t j = i - 3; j <= i; ++j) {
                out_lit[2 * j] = (out[j] & 15) == 15 ? words[r++] : 0xFFFF;
                out_lit[2 * j + 1] = (out[j] >> 4) == 15 ? words[r++] : 0xFFFF;
            }
    }
    *state_end = x;
    return r;
}
