/*
 * sfe_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded CPU oracle for the hot path of arxiv/paper_2606_06811
 * ("Dependencies and Dataflow in Seed-Filter-Extend Pipelines"): LASTZ-style serial
 * Y-drop gapped extension with in-order containment skipping (Algorithm 1)
 * and its speculative, batched restatement (Algorithm 3).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this file.  It shares no code, header, table or constant with the CUDA path
 * (paper_2606_06811_b200/csrc, include/sfe.h); it defines its own structs.
 *
 * The paper names the operations but states none of the recurrences, thresholds or
 * tie-breaks (PAPER.md:59, 203 only name "YDropExtension"); every rule below is a reading
 * fixed in SURVEY.md section 8(c) (R1..R29) and restated in DESIGN.md.  Each function
 * cites the rule / passage it follows.  Everything is written as the definition: row-major
 * loops over explicit cells, no blocking, no fusion, no reordering.
 *
 * Pins (tests/test_oracle_pins.py): SURVEY Appendix A worked examples (tests/golden),
 * ydrop = infinity against a brute-force full Gotoh DP (10^5 trials) and cell by cell against an
 * independent numpy DP, closed forms (incl. lag > n == constant threshold), CIGAR rescoring and
 * the other invariants of SURVEY 8(c) P1..P7, hand-worked tie-break examples for R11 (E / F open
 * on ties, E over F), the four closed box edges of R17, the mirrored query limits of R15, the
 * matrix orientation [query][target] and tau's inclusiveness.  Single-token mutations of every
 * rule turn a pin red, except three that are provably equivalent.
 * No function here is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define OSFE_NEG (-(1 << 30))          /* "minus infinity" for dead / non-existent predecessors */
#define OSFE_YDROP_INF 0x7fffffff      /* R27: pruning disabled                                  */

/* op codes of a run-length edit script (R12): M = aligned pair, I = query base vs gap,
 * D = target base vs gap.  An op word is (len << 4) | code. */
enum { OSFE_M = 0, OSFE_I = 1, OSFE_D = 2 };

typedef struct {
    int32_t sub[4][4];      /* substitution scores, rows/cols A,C,G,T [query][target]          */
    int32_t n_score;        /* R13: score of any pair with N on either side                     */
    int32_t gap_open;       /* R2: a gap of length k costs gap_open + k * gap_extend            */
    int32_t gap_extend;
    int32_t ydrop;          /* R5; OSFE_YDROP_INF = no pruning (R27)                            */
    int32_t prune_lag;      /* R4: row lag Lambda of the "best so far" used by the threshold    */
    int32_t min_score;      /* R16: tau of Alg. 1 line 9 / Alg. 3 line 12                       */
} osfe_scoring;

typedef struct {
    int32_t score;          /* best = H(end_i, end_j) >= 0 (R8)                                 */
    int64_t end_i, end_j;   /* argbest: rows = query bases consumed, cols = target bases (R3)   */
    int64_t cells;          /* R28: sum over rows of (last alive col - first alive col + 1)     */
    int64_t rows;           /* number of rows that had an alive cell                            */
    int64_t max_width;      /* max over rows of (last alive - first alive + 1)                  */
    int64_t n_ops;          /* run-length ops of the traceback, origin -> end order             */
} osfe_half;

static int32_t imax(int32_t a, int32_t b) { return a > b ? a : b; }
/* subtract a cost from a value that may be "minus infinity" */
static int32_t sub_neg(int32_t v, int32_t c) { return v <= OSFE_NEG ? OSFE_NEG : v - c; }

/* R13: score of query code a vs target code b; codes 0..3 = A,C,G,T, 4 = N. */
static int32_t pair_score(const osfe_scoring *sc, uint8_t a, uint8_t b)
{
    if (a > 3 || b > 3) return sc->n_score;
    return sc->sub[a][b];
}

/* ------------------------------------------------------------------------------------------
 * One-sided Y-drop extension (SURVEY 8(c) "One-sided extension ext(q[0..n), t[0..m))";
 * PAPER.md:59 "YDropExtension", "when the alignment score drops below a
 * specific threshold").
 *
 * Rows i = 0..n are query bases consumed, columns j = 0..m target bases consumed (R3).
 * Three-state Gotoh (R1), visited in row-major order; a cell is alive iff it has an alive
 * predecessor and H >= T (R5); dead cells contribute OSFE_NEG on every edge (R6); best is the
 * first maximum in row-major order (R7); origin H(0,0)=0 (R8); stop after the first row with
 * no alive cell.  Threshold (R4): T = B - ydrop, with
 *     lag == 0 : B = best over alive cells preceding (i,j) in row-major order,
 *     lag >= 1 : B = best over alive cells in rows <= i - lag (0 if i < lag).
 * Pointers (R11): one byte per cell: bits 0-1 H source (0 M, 1 E, 2 F; priority M > E > F),
 * bit 2 = E was opened from H(i-1,j) (H-(O+X) >= E-X), bit 3 = F was opened from H(i,j-1).
 *
 * q, t: code arrays (0..3, 4 = N) already oriented so that index 0 is the base next to the
 * anchor.  ops (may be NULL) receives up to ops_cap run-length ops in origin -> end order;
 * out->n_ops is the number needed.  Returns 0, or -1 if out of memory.
 * ------------------------------------------------------------------------------------------ */
static int ext_onesided_cells(const uint8_t *q, int64_t n, const uint8_t *t, int64_t m,
                              const osfe_scoring *sc, osfe_half *out, uint32_t **ops_out,
                              int32_t *cellH, uint8_t *cellA)
{
    const int32_t O = sc->gap_open, X = sc->gap_extend, OX = O + X;
    const int inf = (sc->ydrop == OSFE_YDROP_INF);
    const int64_t lag = sc->prune_lag;

    /* previous row: columns [pL, pR] hold H, E, alive; outside that range every cell is dead */
    int64_t cap = 1024;
    int32_t *Hp = malloc(cap * sizeof *Hp), *Ep = malloc(cap * sizeof *Ep);
    int32_t *Hc = malloc(cap * sizeof *Hc), *Ec = malloc(cap * sizeof *Ec);
    uint8_t *Ap = malloc(cap), *Ac = malloc(cap);
    int64_t pL = 0, pR = -1, pW0 = 0;        /* pW0: column of index 0 of the previous-row arrays */

    /* per-row traceback storage */
    int64_t rcap = 1024, nrows = 0;
    int64_t *row_off = malloc(rcap * sizeof *row_off);   /* offset of the row's bytes in ptr[] */
    int64_t *row_c0 = malloc(rcap * sizeof *row_c0);     /* first stored column of the row      */
    int32_t *best_upto = malloc(rcap * sizeof *best_upto); /* best over alive cells in rows <= r */
    int64_t pcap = 1 << 16, pused = 0;
    uint8_t *ptr = malloc(pcap);
    if (!Hp || !Ep || !Hc || !Ec || !Ap || !Ac || !row_off || !row_c0 || !best_upto || !ptr) return -1;

    int32_t best = 0; int64_t bi = 0, bj = 0;
    int64_t cells = 0, rows_alive = 0, max_width = 0;

    for (int64_t i = 0; i <= n; i++) {
        const int64_t js = (i == 0) ? 0 : pL;            /* no alive predecessor left of pL */
        if (i > 0 && js > m) break;
        if (nrows == rcap) {
            rcap *= 2;
            row_off = realloc(row_off, rcap * sizeof *row_off);
            row_c0 = realloc(row_c0, rcap * sizeof *row_c0);
            best_upto = realloc(best_upto, rcap * sizeof *best_upto);
            if (!row_off || !row_c0 || !best_upto) return -1;
        }
        row_off[nrows] = pused; row_c0[nrows] = js;

        /* R4, lag >= 1: the threshold is the same for the whole row */
        int32_t B_row = 0;
        if (lag >= 1 && i - lag >= 0) B_row = best_upto[i - lag];

        int64_t cL = -1, cR = -1;                         /* first / last alive column of row i */
        int32_t Fprev = OSFE_NEG;                         /* F(i, j-1) */
        int64_t j;
        for (j = js; j <= m; j++) {
            const int64_t k = j - js;                     /* index in the current-row arrays */
            if (k >= cap) {
                cap *= 2;
                Hp = realloc(Hp, cap * sizeof *Hp); Ep = realloc(Ep, cap * sizeof *Ep);
                Hc = realloc(Hc, cap * sizeof *Hc); Ec = realloc(Ec, cap * sizeof *Ec);
                Ap = realloc(Ap, cap); Ac = realloc(Ac, cap);
                if (!Hp || !Ep || !Hc || !Ec || !Ap || !Ac) return -1;
            }
            int32_t H, E, F; uint8_t p = 0; int alive;
            if (i == 0 && j == 0) {                       /* R8: origin */
                H = 0; E = OSFE_NEG; F = OSFE_NEG; alive = 1;
            } else {
                const int up = (i >= 1 && j >= pL && j <= pR && Ap[j - pW0]);
                const int dg = (i >= 1 && j - 1 >= pL && j - 1 <= pR && Ap[j - 1 - pW0]);
                const int lf = (j - 1 >= js && Ac[k - 1]);
                int32_t M = OSFE_NEG;
                E = OSFE_NEG; F = OSFE_NEG;
                if (up) {                                 /* 'I': consumes a query base */
                    const int32_t open = Hp[j - pW0] - OX, ext = sub_neg(Ep[j - pW0], X);
                    E = imax(open, ext);
                    if (open >= ext) p |= 4;              /* R11: open wins ties */
                }
                if (lf) {                                 /* 'D': consumes a target base */
                    const int32_t open = Hc[k - 1] - OX, ext = sub_neg(Fprev, X);
                    F = imax(open, ext);
                    if (open >= ext) p |= 8;
                }
                if (dg) M = Hp[j - 1 - pW0] + pair_score(sc, q[i - 1], t[j - 1]);
                H = imax(M, imax(E, F));
                if (H <= OSFE_NEG) {
                    alive = 0;                            /* no alive predecessor */
                } else {
                    if (H == M) p |= 0; else if (H == E) p |= 1; else p |= 2;   /* M > E > F */
                    if (inf) alive = 1;                   /* R27 */
                    else {
                        const int32_t B = (lag == 0) ? best : B_row;            /* R4 */
                        alive = (H >= B - sc->ydrop);                           /* R5 */
                    }
                }
            }
            Hc[k] = H; Ec[k] = E; Ac[k] = (uint8_t)alive; Fprev = F;
            if (cellH) cellH[i * (m + 1) + j] = H;        /* inspection only (pin P5): no effect on the DP */
            if (cellA) cellA[i * (m + 1) + j] = (uint8_t)alive;
            if (pused == pcap) { pcap *= 2; ptr = realloc(ptr, pcap); if (!ptr) return -1; }
            ptr[pused++] = p;
            if (alive) {
                if (cL < 0) cL = j;
                cR = j;
                if (H > best) { best = H; bi = i; bj = j; }                     /* R7: strict */
            } else if (j > pR + 1) {
                /* beyond the last column the previous row can feed, a dead cell ends the row:
                   every later cell has only the (dead) left neighbour as predecessor */
                break;
            }
        }
        nrows++;
        if (cL < 0) { nrows--; pused = row_off[nrows]; break; }   /* first row with no alive cell */
        best_upto[i] = best;
        cells += cR - cL + 1; rows_alive++;
        if (cR - cL + 1 > max_width) max_width = cR - cL + 1;
        /* current row becomes previous row */
        { int32_t *x = Hp; Hp = Hc; Hc = x; x = Ep; Ep = Ec; Ec = x; uint8_t *y = Ap; Ap = Ac; Ac = y; }
        pW0 = js; pL = cL; pR = cR;
    }

    out->score = best; out->end_i = bi; out->end_j = bj;
    out->cells = cells; out->rows = rows_alive; out->max_width = max_width;

    /* R11 traceback state machine from argbest to the origin, collecting ops end -> origin */
    int64_t nops = 0, ocap = 64;
    uint32_t *rev = malloc(ocap * sizeof *rev);
    if (!rev) return -1;
    {
        int64_t i = bi, j = bj; int state = 0;            /* 0 = H, 1 = E, 2 = F */
        int cur = -1; int64_t run = 0;
        while (!(i == 0 && j == 0 && state == 0)) {
            const uint8_t p = ptr[row_off[i] + (j - row_c0[i])];
            int op = -1;
            if (state == 0) {
                const int src = p & 3;
                if (src == 0) { op = OSFE_M; i--; j--; }
                else state = src;                          /* same cell, gap state */
            } else if (state == 1) {
                op = OSFE_I; state = (p & 4) ? 0 : 1; i--;
            } else {
                op = OSFE_D; state = (p & 8) ? 0 : 2; j--;
            }
            if (op >= 0) {
                if (op == cur) run++;
                else {
                    if (cur >= 0) {
                        if (nops == ocap) { ocap *= 2; rev = realloc(rev, ocap * sizeof *rev); if (!rev) return -1; }
                        rev[nops++] = (uint32_t)(run << 4) | (uint32_t)cur;
                    }
                    cur = op; run = 1;
                }
            }
        }
        if (cur >= 0) {
            if (nops == ocap) { ocap *= 2; rev = realloc(rev, ocap * sizeof *rev); if (!rev) return -1; }
            rev[nops++] = (uint32_t)(run << 4) | (uint32_t)cur;
        }
    }
    out->n_ops = nops;
    if (ops_out) {                                        /* origin -> end order; caller frees */
        uint32_t *fw = malloc((size_t)(nops + 1) * sizeof *fw);
        if (!fw) return -1;
        for (int64_t k = 0; k < nops; k++) fw[k] = rev[nops - 1 - k];
        *ops_out = fw;
    }

    free(rev); free(Hp); free(Ep); free(Hc); free(Ec); free(Ap); free(Ac);
    free(row_off); free(row_c0); free(best_upto); free(ptr);
    return 0;
}

static int ext_onesided_alloc(const uint8_t *q, int64_t n, const uint8_t *t, int64_t m,
                              const osfe_scoring *sc, osfe_half *out, uint32_t **ops_out)
{
    return ext_onesided_cells(q, n, t, m, sc, out, ops_out, NULL, NULL);
}

/* The same extension, also writing every VISITED cell's H and alive flag into dense (n+1) x (m+1)
 * arrays the caller pre-filled (cells never visited keep the caller's fill).  Used only by pin P5
 * ("every alive cell's H is <= its unpruned Gotoh value"). */
int osfe_ext_onesided_cells(const uint8_t *q, int64_t n, const uint8_t *t, int64_t m,
                            const osfe_scoring *sc, osfe_half *out, int32_t *cellH, uint8_t *cellA)
{
    return ext_onesided_cells(q, n, t, m, sc, out, NULL, cellH, cellA);
}

int osfe_ext_onesided(const uint8_t *q, int64_t n, const uint8_t *t, int64_t m,
                      const osfe_scoring *sc, osfe_half *out, uint32_t *ops, int64_t ops_cap)
{
    uint32_t *fw = NULL;
    const int rc = ext_onesided_alloc(q, n, t, m, sc, out, ops ? &fw : NULL);
    if (rc) return rc;
    if (ops) { for (int64_t k = 0; k < out->n_ops && k < ops_cap; k++) ops[k] = fw[k]; free(fw); }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Brute-force full Gotoh DP over the whole (n+1) x (m+1) rectangle, no pruning: the textbook
 * recurrence (R1, R2, R8) with best = first maximum over all cells in row-major order.
 * Independent of osfe_ext_onesided (different storage, no alive logic); used as pin P2.
 * ------------------------------------------------------------------------------------------ */
int osfe_gotoh_bruteforce(const uint8_t *q, int64_t n, const uint8_t *t, int64_t m,
                          const osfe_scoring *sc, int32_t *score, int64_t *end_i, int64_t *end_j)
{
    const int64_t W = m + 1;
    const int64_t MINF = -(1LL << 40);
    int64_t *H = malloc((n + 1) * W * sizeof *H), *E = malloc((n + 1) * W * sizeof *E),
            *F = malloc((n + 1) * W * sizeof *F);
    if (!H || !E || !F) return -1;
    const int64_t OX = sc->gap_open + sc->gap_extend, X = sc->gap_extend;
    int64_t best = 0, bi = 0, bj = 0;
    for (int64_t i = 0; i <= n; i++)
        for (int64_t j = 0; j <= m; j++) {
            int64_t h, e = MINF, f = MINF, d = MINF;
            if (i == 0 && j == 0) h = 0;
            else {
                if (i > 0) { int64_t a = H[(i - 1) * W + j] - OX, b = E[(i - 1) * W + j] - X; e = a > b ? a : b; }
                if (j > 0) { int64_t a = H[i * W + j - 1] - OX, b = F[i * W + j - 1] - X; f = a > b ? a : b; }
                if (i > 0 && j > 0) d = H[(i - 1) * W + j - 1] + pair_score(sc, q[i - 1], t[j - 1]);
                h = d; if (e > h) h = e; if (f > h) h = f;
            }
            H[i * W + j] = h; E[i * W + j] = e; F[i * W + j] = f;
            if (h > best) { best = h; bi = i; bj = j; }
        }
    *score = (int32_t)best; *end_i = bi; *end_j = bj;
    free(H); free(E); free(F);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Rescoring rule of R12 / pin P4: M pairs score pair_score, every emitted run of I or D of
 * length k costs gap_open + k * gap_extend.  Also returns the bases consumed.
 * ------------------------------------------------------------------------------------------ */
int64_t osfe_rescore(const uint8_t *q, const uint8_t *t, const uint32_t *ops, int64_t n_ops,
                     const osfe_scoring *sc, int64_t *q_used, int64_t *t_used)
{
    int64_t s = 0, i = 0, j = 0;
    for (int64_t k = 0; k < n_ops; k++) {
        const int64_t len = ops[k] >> 4; const int op = ops[k] & 15;
        if (op == OSFE_M) { for (int64_t x = 0; x < len; x++) s += pair_score(sc, q[i + x], t[j + x]); i += len; j += len; }
        else if (op == OSFE_I) { s -= sc->gap_open + len * (int64_t)sc->gap_extend; i += len; }
        else { s -= sc->gap_open + len * (int64_t)sc->gap_extend; j += len; }
    }
    *q_used = i; *t_used = j;
    return s;
}

/* ------------------------------------------------------------------------------------------
 * Sequence packing (R13, R14): ASCII -> code (A0 C1 G2 T3, case-insensitive, anything else N).
 * Planes: 2-bit codes (base k in byte k/4, bits 2(k%4)..2(k%4)+1; N stored as 0) and 1-bit
 * N mask (base k in byte k/8, bit k%8).  Reverse-complement planes hold 3-code in reversed
 * order with the mask reversed.
 * ------------------------------------------------------------------------------------------ */
static uint8_t ascii_code(char c)
{
    switch (c) {
    case 'A': case 'a': return 0;
    case 'C': case 'c': return 1;
    case 'G': case 'g': return 2;
    case 'T': case 't': return 3;
    default: return 4;
    }
}

void osfe_codes(const char *ascii, int64_t len, uint8_t *codes)
{
    for (int64_t k = 0; k < len; k++) codes[k] = ascii_code(ascii[k]);
}

void osfe_revcomp_codes(const uint8_t *codes, int64_t len, uint8_t *rc)
{
    for (int64_t k = 0; k < len; k++) {
        const uint8_t c = codes[len - 1 - k];
        rc[k] = c > 3 ? 4 : (uint8_t)(3 - c);
    }
}

void osfe_pack(const char *ascii, int64_t len, uint8_t *codes2, uint8_t *nmask,
               uint8_t *rc_codes2, uint8_t *rc_nmask)
{
    memset(codes2, 0, (size_t)((len + 3) / 4)); memset(nmask, 0, (size_t)((len + 7) / 8));
    if (rc_codes2) memset(rc_codes2, 0, (size_t)((len + 3) / 4));
    if (rc_nmask) memset(rc_nmask, 0, (size_t)((len + 7) / 8));
    for (int64_t k = 0; k < len; k++) {
        const uint8_t c = ascii_code(ascii[k]);
        const int64_t r = len - 1 - k;
        if (c > 3) {
            nmask[k / 8] |= (uint8_t)(1u << (k % 8));
            if (rc_nmask) rc_nmask[r / 8] |= (uint8_t)(1u << (r % 8));
        } else {
            codes2[k / 4] |= (uint8_t)(c << (2 * (k % 4)));
            if (rc_codes2) rc_codes2[r / 4] |= (uint8_t)((3 - c) << (2 * (r % 4)));
        }
    }
}

/* ------------------------------------------------------------------------------------------
 * Two-sided extension of one anchor (SURVEY 8(c) "Two-sided"; R9, R10, R12, R15).
 * T, Q: code arrays of the whole target and of the query IN THE ANCHOR'S STRAND FRAME (for
 * strand -1 the caller passes the reverse-complemented query and limits in that frame).
 * forward  = ext(Q[qpos..q_end), T[tpos..t_end));
 * backward = ext(reverse(Q[q_begin..qpos)), reverse(T[t_begin..tpos))).
 * ops: backward runs in reversed order, then forward runs; never merged across the junction.
 * ------------------------------------------------------------------------------------------ */
typedef struct {
    int32_t score, score_fwd, score_bwd;
    int64_t tstart, tend, qstart, qend;     /* box, corner coordinates */
    int64_t n_ops, n_ops_back;
    int64_t cells, cells_fwd, cells_bwd;
    int64_t rows_fwd, rows_bwd, max_width;
} osfe_result;

int osfe_extend_anchor(const uint8_t *T, int64_t t_begin, int64_t t_end,
                       const uint8_t *Q, int64_t q_begin, int64_t q_end,
                       int64_t tpos, int64_t qpos, const osfe_scoring *sc,
                       osfe_result *res, uint32_t *ops, int64_t ops_cap)
{
    osfe_half f, b;
    uint32_t *fo = NULL, *bo = NULL;
    /* forward */
    const int64_t nf = q_end - qpos, mf = t_end - tpos;
    if (nf < 0 || mf < 0 || qpos < q_begin || tpos < t_begin) return -2;
    if (ext_onesided_alloc(Q + qpos, nf, T + tpos, mf, sc, &f, ops ? &fo : NULL)) return -1;
    /* backward: explicit reversed copies (R9) */
    const int64_t nb = qpos - q_begin, mb = tpos - t_begin;
    uint8_t *qr = malloc((size_t)(nb > 0 ? nb : 1)), *tr = malloc((size_t)(mb > 0 ? mb : 1));
    if (!qr || !tr) return -1;
    for (int64_t k = 0; k < nb; k++) qr[k] = Q[qpos - 1 - k];
    for (int64_t k = 0; k < mb; k++) tr[k] = T[tpos - 1 - k];
    if (ext_onesided_alloc(qr, nb, tr, mb, sc, &b, ops ? &bo : NULL)) return -1;

    res->score_fwd = f.score; res->score_bwd = b.score; res->score = f.score + b.score;
    res->tstart = tpos - b.end_j; res->tend = tpos + f.end_j;
    res->qstart = qpos - b.end_i; res->qend = qpos + f.end_i;
    res->n_ops = f.n_ops + b.n_ops; res->n_ops_back = b.n_ops;
    res->cells_fwd = f.cells; res->cells_bwd = b.cells; res->cells = f.cells + b.cells;
    res->rows_fwd = f.rows; res->rows_bwd = b.rows;
    res->max_width = f.max_width > b.max_width ? f.max_width : b.max_width;

    if (ops) {                                            /* R12: never merged across the junction */
        int64_t w = 0;
        for (int64_t k = b.n_ops - 1; k >= 0 && w < ops_cap; k--) ops[w++] = bo[k];   /* reversed */
        for (int64_t k = 0; k < f.n_ops && w < ops_cap; k++) ops[w++] = fo[k];
        free(fo); free(bo);
    }
    free(qr); free(tr);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Containment predicate (R17, R26; PAPER.md:48 IsContained, PAPER.md:122 IsMasked): the anchor
 * point lies in an accepted bounding box of the same strand, closed intervals.
 * ------------------------------------------------------------------------------------------ */
typedef struct { int64_t tstart, tend, qstart, qend; int32_t strand; } osfe_box;
typedef struct { int64_t tpos, qpos; int32_t pair; int32_t strand; } osfe_anchor;
typedef struct { int64_t t_begin, t_end, q_begin, q_end; } osfe_pair;

static int covered(const osfe_box *acc, int64_t n_acc, const osfe_anchor *a)
{
    for (int64_t k = 0; k < n_acc; k++)
        if (acc[k].strand == a->strand && acc[k].tstart <= a->tpos && a->tpos <= acc[k].tend &&
            acc[k].qstart <= a->qpos && a->qpos <= acc[k].qend)
            return 1;
    return 0;
}

/* strand frame of the query limits: for strand -1 the pair's query interval is mirrored into
 * the reverse-complement frame (R15) */
static void pair_limits(const osfe_pair *p, int32_t strand, int64_t q_len, int64_t *qb, int64_t *qe)
{
    if (strand >= 0) { *qb = p->q_begin; *qe = p->q_end; }
    else { *qb = q_len - p->q_end; *qe = q_len - p->q_begin; }
}

/* ------------------------------------------------------------------------------------------
 * Algorithm 1, the serial loop (SURVEY 8(c) "Serial loop"):
 * state[i] = 0 covered (not extended), 1 kept, 2 below tau (extended, masks nothing: R18).
 * results[i] is filled for every anchor that was extended.  Returns number kept, or < 0.
 * ------------------------------------------------------------------------------------------ */
int64_t osfe_serial_loop(const uint8_t *T, const uint8_t *Q, const uint8_t *Qrc, int64_t q_len,
                         const osfe_pair *pairs, const osfe_anchor *anchors, int64_t n,
                         const osfe_scoring *sc, uint8_t *state, osfe_result *results,
                         int64_t *n_extended, int64_t *cells_extended)
{
    osfe_box *acc = malloc((size_t)(n > 0 ? n : 1) * sizeof *acc);
    int64_t n_acc = 0, next = 0, cells = 0;
    if (!acc) return -1;
    for (int64_t i = 0; i < n; i++) {
        const osfe_anchor *a = &anchors[i];
        if (covered(acc, n_acc, a)) { state[i] = 0; continue; }          /* Alg. 1 line 3 */
        const osfe_pair *p = &pairs[a->pair];
        int64_t qb, qe; pair_limits(p, a->strand, q_len, &qb, &qe);
        osfe_result r;
        if (osfe_extend_anchor(T, p->t_begin, p->t_end, a->strand >= 0 ? Q : Qrc, qb, qe,
                               a->tpos, a->qpos, sc, &r, NULL, 0)) { free(acc); return -1; }
        next++; cells += r.cells;                                        /* Alg. 1 line 8 */
        if (results) results[i] = r;
        if (r.score >= sc->min_score) {                                  /* Alg. 1 lines 9-11 */
            acc[n_acc].tstart = r.tstart; acc[n_acc].tend = r.tend;
            acc[n_acc].qstart = r.qstart; acc[n_acc].qend = r.qend; acc[n_acc].strand = a->strand;
            n_acc++; state[i] = 1;
        } else state[i] = 2;
    }
    if (n_extended) *n_extended = next;
    if (cells_extended) *cells_extended = cells;
    free(acc);
    return n_acc;
}

/* ------------------------------------------------------------------------------------------
 * Algorithm 3, the speculative windowed loop: Phase 1 gathers K anchors not
 * masked by alignments committed in EARLIER windows (R26); Phase 2 extends all of them; Phase 3
 * commits in batch order with the containment test against everything accepted so far (R17).
 * state[] as in the serial loop (anchors skipped in phase 1 are 0).  spec_extended[i] = 1 if
 * anchor i was extended speculatively.  Returns number kept.
 * ------------------------------------------------------------------------------------------ */
int64_t osfe_speculative_loop(const uint8_t *T, const uint8_t *Q, const uint8_t *Qrc, int64_t q_len,
                              const osfe_pair *pairs, const osfe_anchor *anchors, int64_t n,
                              const osfe_scoring *sc, int64_t K, uint8_t *state,
                              uint8_t *spec_extended, int64_t *n_extended, int64_t *cells_extended)
{
    osfe_box *acc = malloc((size_t)(n > 0 ? n : 1) * sizeof *acc);
    int64_t *batch = malloc((size_t)(K > 0 ? K : 1) * sizeof *batch);
    osfe_result *ext = malloc((size_t)(K > 0 ? K : 1) * sizeof *ext);
    int64_t n_acc = 0, next = 0, cells = 0, j = 0;
    if (!acc || !batch || !ext || K < 1) return -1;
    for (int64_t i = 0; i < n; i++) { state[i] = 0; if (spec_extended) spec_extended[i] = 0; }
    while (j < n) {
        int64_t nb = 0;
        while (nb < K && j < n) {                                        /* Phase 1 */
            if (!covered(acc, n_acc, &anchors[j])) batch[nb++] = j;
            j++;
        }
        for (int64_t b = 0; b < nb; b++) {                               /* Phase 2 */
            const osfe_anchor *a = &anchors[batch[b]];
            const osfe_pair *p = &pairs[a->pair];
            int64_t qb, qe; pair_limits(p, a->strand, q_len, &qb, &qe);
            if (osfe_extend_anchor(T, p->t_begin, p->t_end, a->strand >= 0 ? Q : Qrc, qb, qe,
                                   a->tpos, a->qpos, sc, &ext[b], NULL, 0)) return -1;
            next++; cells += ext[b].cells;
            if (spec_extended) spec_extended[batch[b]] = 1;
        }
        for (int64_t b = 0; b < nb; b++) {                               /* Phase 3 */
            const int64_t i = batch[b];
            if (covered(acc, n_acc, &anchors[i])) { state[i] = 0; continue; }
            if (ext[b].score >= sc->min_score) {
                acc[n_acc].tstart = ext[b].tstart; acc[n_acc].tend = ext[b].tend;
                acc[n_acc].qstart = ext[b].qstart; acc[n_acc].qend = ext[b].qend;
                acc[n_acc].strand = anchors[i].strand;
                n_acc++; state[i] = 1;
            } else state[i] = 2;
        }
    }
    if (n_extended) *n_extended = next;
    if (cells_extended) *cells_extended = cells;
    free(acc); free(batch); free(ext);
    return n_acc;
}

/* ------------------------------------------------------------------------------------------
 * Resolve only (phase 3 given finished extensions): kept(i) = score_i >= tau and no kept j < i
 * of the same strand has box_j containing the anchor point of i.  Anchors tested against the
 * `accepted` boxes from earlier windows first (R26).  state as above.
 * ------------------------------------------------------------------------------------------ */
int64_t osfe_resolve(const osfe_anchor *anchors, const osfe_result *results, int64_t n,
                     int32_t min_score, osfe_box *accepted, int64_t n_accepted, int64_t accepted_cap,
                     uint8_t *state)
{
    for (int64_t i = 0; i < n; i++) {
        if (covered(accepted, n_accepted, &anchors[i])) { state[i] = 0; continue; }
        if (results[i].score >= min_score) {
            if (n_accepted >= accepted_cap) return -1;
            accepted[n_accepted].tstart = results[i].tstart; accepted[n_accepted].tend = results[i].tend;
            accepted[n_accepted].qstart = results[i].qstart; accepted[n_accepted].qend = results[i].qend;
            accepted[n_accepted].strand = anchors[i].strand;
            n_accepted++; state[i] = 1;
        } else state[i] = 2;
    }
    return n_accepted;
}

/* struct sizes, so that the ctypes mirror in sfe_oracle.py can assert its layout */
int64_t osfe_sizeof(int which)
{
    switch (which) {
    case 0: return sizeof(osfe_scoring);
    case 1: return sizeof(osfe_half);
    case 2: return sizeof(osfe_result);
    case 3: return sizeof(osfe_box);
    case 4: return sizeof(osfe_anchor);
    case 5: return sizeof(osfe_pair);
    default: return -1;
    }
}
