/*
 * lpf_oracle.c -- plain CPU oracle for the lineal path function L2 of a periodic
 * two-phase pixel image (Havelka, Kucerova, Sykora, arXiv 1601.04359).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code with the CUDA library under paper_1601_04359_b200/csrc and must
 * never be imported from there.
 *
 * What it computes is the plain definition, shaped like the paper's Alg. 1
 * ("for seg / for transl / for pix ... if A[...] != phase break"):
 *
 *   count_phi(v) = #{ (x,y) in [0,W)x[0,H) :
 *                     I[(y+b) mod H][(x+a) mod W] == phi  for all (a,b) in P_v }
 *
 * with  L2_phi(v) = count_phi(v) / (W*H)   (Eq. 6's 1/(WH) normalisation, PAPER.md:99;
 * Eq. 10 L2(0) = phi).  No bit packing, no trie, no SIMD, no symmetry
 * shortcut unless the caller asks for the mirrored half (Eq. 12).
 *
 * Readings of the paper taken here (all listed in DESIGN.md "Readings"):
 *   D1  |P_v| = max(|dx|,|dy|) + 1, both end pixels included (Eq. 15's max(i,j)).
 *   D2  v in the canonical half D (Eq. 13: dy>0, or dy==0 and dx>=0):
 *       Bresenham [20] from (0,0) to v in the incremental-error form below; ties go to
 *       the larger |minor| coordinate; signs applied after.  The paper is silent on ties.
 *   D3  v not in D:  P_v = reverse(P_{-v}) + v, the same pixel set as the canonical
 *       segment ("the line segment x1x2 is identical to x2x1").
 *   S2  x <-> column <-> W,  y <-> row <-> H  (Eq. 6: x%W, y%H).
 *   S3  Alg. 1 loops pix = 0..D[seg]-1 and counts a hit iff no break.
 *   S8  a pixel is "in phase phi" iff its byte equals phi (Alg. 1 line 4).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Eq. 15-17 and |D| closed forms, the worked
 * paths/image in tests/golden/, stripes and run-length closed forms, scipy erosion,
 * numpy FFT autocorrelation for |P_v| = 2 (Eq. 6/7), brute force by whole-array
 * roll-and-AND on tiny images, Eq. 10/12 invariants, Bernoulli statistics.
 * lpf_oracle_counts_masked (L2~): all-ones mask = lpf_oracle_counts_list, additivity over disjoint
 * masks, one-pixel masks vs the definition.  lpf_oracle_s2_counts (Eq. 6): numpy FFT form of Eq. 7, S2(0) = phase
 * count, point symmetry, equality with the lineal-path counts for the 8 neighbours (|P_v| = 2).
 * lpf_oracle_counts_sum (ensemble over a stack): one image = lpf_oracle_counts, additive over a split of
 * the stack, k copies of the worked image = k times its golden counts, Eq. 10 summed (centre = phase pixels of the stack).
 * lpf_oracle_splitmix64 / lpf_oracle_propose (modification operator, reading A7): the published SplitMix64 test vectors;
 * every generated pair has different bytes and (policy 2) two interfacial pixels, checked with numpy; uniform over the
 * qualifying pixels (chi-square); the generating chain = the list chain fed with the generated pairs.
 * lpf_oracle_anneal (Alg. 3): the Metropolis threshold at finite T against exact rationals computed in the test, volume fractions preserved, E tracked = Eq. 19 of the final image re-evaluated, a huge
 * T accepts every move (final image = all swaps applied, temperature levels = floor(N / s_max)), a tiny T never lets E
 * grow, the local-delta form equals the literal re-evaluation form decision by decision.
 * Parity with the AUTHORS' numbers is unpinned: the paper prints no L2 value.
 *
 * Build:  gcc -O2 -fopenmp -shared -fPIC -o liblpf_oracle.so lpf_oracle.c
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

static int iabs_(int v) { return v < 0 ? -v : v; }
static int imax_(int a, int b) { return a > b ? a : b; }
static int sgn_(int v) { return (v > 0) - (v < 0); }
static int pmod_(int a, int n) { int r = a % n; return r < 0 ? r + n : r; }

/* Is v in the canonical half-plane D of Eq. 13? */
int lpf_oracle_in_half(int dx, int dy) { return dy > 0 || (dy == 0 && dx >= 0); }

/* D2: Bresenham, incremental error form, for v in D.  xy = [len][2] (x then y). */
static int canonical_path_(int dx, int dy, int16_t *xy)
{
    int ax = iabs_(dx), ay = iabs_(dy), sx = sgn_(dx), sy = sgn_(dy);
    int x = 0, y = 0, n = 0;
    xy[0] = 0; xy[1] = 0; n = 1;
    if (ax >= ay) {                       /* x-major: one pixel per x step */
        int e = ax;
        for (int k = 0; k < ax; ++k) {
            x += sx;
            e += 2 * ay;
            if (e >= 2 * ax) { y += sy; e -= 2 * ax; }
            xy[2 * n] = (int16_t)x; xy[2 * n + 1] = (int16_t)y; ++n;
        }
    } else {                              /* y-major: one pixel per y step */
        int e = ay;
        for (int k = 0; k < ay; ++k) {
            y += sy;
            e += 2 * ax;
            if (e >= 2 * ay) { x += sx; e -= 2 * ay; }
            xy[2 * n] = (int16_t)x; xy[2 * n + 1] = (int16_t)y; ++n;
        }
    }
    return n;
}

/* P_v for ANY v (D2 for v in D, D3 otherwise).  xy must hold max(|dx|,|dy|)+1 pairs.
 * Returns |P_v|. */
int lpf_oracle_path(int dx, int dy, int16_t *xy)
{
    if (lpf_oracle_in_half(dx, dy)) return canonical_path_(dx, dy, xy);
    int n = canonical_path_(-dx, -dy, xy);            /* P_{-v} */
    for (int i = 0, j = n - 1; i < j; ++i, --j) {      /* reverse the order */
        int16_t tx = xy[2 * i], ty = xy[2 * i + 1];
        xy[2 * i] = xy[2 * j]; xy[2 * i + 1] = xy[2 * j + 1];
        xy[2 * j] = tx; xy[2 * j + 1] = ty;
    }
    for (int i = 0; i < n; ++i) {                      /* translate by v */
        xy[2 * i] = (int16_t)(xy[2 * i] + dx);
        xy[2 * i + 1] = (int16_t)(xy[2 * i + 1] + dy);
    }
    return n;
}

/* Alg. 1 lines 2-10 for ONE segment: translate over every start pixel, compare, count. */
static int64_t count_one_(const uint8_t *img, int H, int W, int phase,
                          const int16_t *xy, int n)
{
    int64_t hits = 0;
    for (int y = 0; y < H; ++y) {                       /* "transl" */
        for (int x = 0; x < W; ++x) {
            int pix;
            for (pix = 0; pix < n; ++pix) {             /* "pix" */
                int xx = pmod_(x + xy[2 * pix], W);
                int yy = pmod_(y + xy[2 * pix + 1], H);
                if (img[(size_t)yy * W + xx] != phase) break;
            }
            if (pix == n) ++hits;                       /* Alg. 1 lines 8-9 */
        }
    }
    return hits;
}

/* Counts for a caller-given list of vectors vecs = [n][2] (dx,dy); out[n].
 * threads <= 0 means "all the OpenMP runtime gives". Returns the threads used. */
int lpf_oracle_counts_list(const uint8_t *img, int H, int W, int phase,
                           const int32_t *vecs, int64_t n, int64_t *out, int threads)
{
    int used = 1;
#ifdef _OPENMP
    if (threads <= 0) threads = omp_get_max_threads();
    used = threads;
#else
    (void)threads;
#endif
#pragma omp parallel num_threads(used)
    {
        int16_t *xy = NULL; int cap = 0;
#pragma omp for schedule(dynamic, 4)
        for (int64_t i = 0; i < n; ++i) {
            int dx = vecs[2 * i], dy = vecs[2 * i + 1];
            int need = imax_(iabs_(dx), iabs_(dy)) + 1;
            if (need > cap) { free(xy); cap = need; xy = (int16_t *)malloc(sizeof(int16_t) * 2 * (size_t)cap); }
            int len = lpf_oracle_path(dx, dy, xy);
            out[i] = count_one_(img, H, W, phase, xy, len);
        }
        free(xy);
    }
    return used;
}

/* The whole template |dx|,|dy| <= m: counts[(dy+m)*(2m+1) + (dx+m)].
 *   full_template = 1: every one of the (2m+1)^2 vectors is evaluated on its own path
 *                      (nothing mirrored) -- used to SHOW Eq. 12 rather than assume it;
 *   full_template = 0: only v in D is evaluated, counts[-v] = counts[v].
 * Returns the threads used. */
int lpf_oracle_counts(const uint8_t *img, int H, int W, int phase, int m,
                      int64_t *counts, int full_template, int threads)
{
    int S = 2 * m + 1;
    int64_t nvec = 0;
    int32_t *vecs = (int32_t *)malloc(sizeof(int32_t) * 2 * (size_t)S * S);
    int64_t *tmp = (int64_t *)malloc(sizeof(int64_t) * (size_t)S * S);
    for (int dy = -m; dy <= m; ++dy)
        for (int dx = -m; dx <= m; ++dx)
            if (full_template || lpf_oracle_in_half(dx, dy)) {
                vecs[2 * nvec] = dx; vecs[2 * nvec + 1] = dy; ++nvec;
            }
    int used = lpf_oracle_counts_list(img, H, W, phase, vecs, nvec, tmp, threads);
    for (int64_t i = 0; i < nvec; ++i) {
        int dx = vecs[2 * i], dy = vecs[2 * i + 1];
        counts[(size_t)(dy + m) * S + (dx + m)] = tmp[i];
        if (!full_template)
            counts[(size_t)(-dy + m) * S + (-dx + m)] = tmp[i];
    }
    free(vecs); free(tmp);
    return used;
}

/* Ensemble descriptor of a stack of B images of one size (the descriptor of the specimen is "averaged
 * over 100 slices"): sum_out[v] = sum_b count(image_b, v); the ensemble average of L2 is sum_out / (B*W*H), one division
 * by the caller.  Plain loop over the images, each evaluated on its own by lpf_oracle_counts (canonical half + Eq. 12). */
void lpf_oracle_counts_sum(const uint8_t *imgs, int B, int H, int W, int phase, int m,
                           int64_t *sum_out, int threads)
{
    int S = 2 * m + 1;
    size_t K = (size_t)S * S;
    int64_t *one = (int64_t *)malloc(sizeof(int64_t) * K);
    for (size_t k = 0; k < K; ++k) sum_out[k] = 0;
    for (int b = 0; b < B; ++b) {
        lpf_oracle_counts(imgs + (size_t)b * H * W, H, W, phase, m, one, 0, threads);
        for (size_t k = 0; k < K; ++k) sum_out[k] += one[k];
    }
    free(one);
}

/* Eq. 14 / Eq. 19 on integer counts: sum_k (c_k - t_k)^2, exact.
 * (e = sse / (W*H)^2 is one IEEE division done by the caller.) */
uint64_t lpf_oracle_sse(const int64_t *counts, const int64_t *target, int64_t K)
{
    uint64_t s = 0;
    for (int64_t k = 0; k < K; ++k) {
        int64_t d = counts[k] - target[k];
        s += (uint64_t)(d * d);
    }
    return s;
}

/* Two-pixel swap ("interchanging two randomly chosen pixels from different
 * phases"), BY DEFINITION: delta(v) = count(I', v) - count(I, v) with I' = I after the two
 * pixels (xp,yp) and (xq,yq) exchange their bytes.  Full re-evaluation, twice. */
int lpf_oracle_swap_delta_full(const uint8_t *img, int H, int W, int phase, int m,
                               int xp, int yp, int xq, int yq, int32_t *delta, int threads)
{
    int S = 2 * m + 1;
    size_t K = (size_t)S * S;
    uint8_t *img2 = (uint8_t *)malloc((size_t)H * W);
    int64_t *c0 = (int64_t *)malloc(sizeof(int64_t) * K);
    int64_t *c1 = (int64_t *)malloc(sizeof(int64_t) * K);
    memcpy(img2, img, (size_t)H * W);
    uint8_t t = img2[(size_t)yp * W + xp];
    img2[(size_t)yp * W + xp] = img2[(size_t)yq * W + xq];
    img2[(size_t)yq * W + xq] = t;
    int used = lpf_oracle_counts(img, H, W, phase, m, c0, 0, threads);
    lpf_oracle_counts(img2, H, W, phase, m, c1, 0, threads);
    for (size_t k = 0; k < K; ++k) delta[k] = (int32_t)(c1[k] - c0[k]);
    free(img2); free(c0); free(c1);
    return used;
}

/* Same delta, restricted to the start pixels whose segment can change: a segment (s,v)
 * differs between I and I' only if it contains p or q, i.e. s = p - P_v[k] or q - P_v[k].
 * Still the definition (each candidate start is tested on I and on I' pixel by pixel);
 * pinned to lpf_oracle_swap_delta_full in tests/test_oracle_swap.py. */
static int seg_in_phase_(const uint8_t *img, int H, int W, int phase,
                         const int16_t *xy, int n, int sx, int sy)
{
    for (int pix = 0; pix < n; ++pix) {
        int xx = pmod_(sx + xy[2 * pix], W);
        int yy = pmod_(sy + xy[2 * pix + 1], H);
        if (img[(size_t)yy * W + xx] != phase) return 0;
    }
    return 1;
}

void lpf_oracle_swap_delta_local(const uint8_t *img, int H, int W, int phase, int m,
                                 int xp, int yp, int xq, int yq, int32_t *delta)
{
    int S = 2 * m + 1;
    uint8_t *img2 = (uint8_t *)malloc((size_t)H * W);
    int16_t *xy = (int16_t *)malloc(sizeof(int16_t) * 2 * (size_t)(m + 1));
    int *sxs = (int *)malloc(sizeof(int) * 2 * (size_t)(m + 1));
    int *sys = (int *)malloc(sizeof(int) * 2 * (size_t)(m + 1));
    memcpy(img2, img, (size_t)H * W);
    uint8_t t = img2[(size_t)yp * W + xp];
    img2[(size_t)yp * W + xp] = img2[(size_t)yq * W + xq];
    img2[(size_t)yq * W + xq] = t;
    for (int dy = -m; dy <= m; ++dy)
        for (int dx = -m; dx <= m; ++dx) {
            int n = lpf_oracle_path(dx, dy, xy);
            int ns = 0;
            /* candidate starts, de-duplicated (p - P_v[k] may equal q - P_v[j]) */
            for (int side = 0; side < 2; ++side)
                for (int k = 0; k < n; ++k) {
                    int sx = pmod_((side ? xq : xp) - xy[2 * k], W);
                    int sy = pmod_((side ? yq : yp) - xy[2 * k + 1], H);
                    int dup = 0;
                    for (int j = 0; j < ns; ++j) if (sxs[j] == sx && sys[j] == sy) { dup = 1; break; }
                    if (!dup) { sxs[ns] = sx; sys[ns] = sy; ++ns; }
                }
            int32_t d = 0;
            for (int j = 0; j < ns; ++j)
                d += seg_in_phase_(img2, H, W, phase, xy, n, sxs[j], sys[j])
                   - seg_in_phase_(img,  H, W, phase, xy, n, sxs[j], sys[j]);
            delta[(size_t)(dy + m) * S + (dx + m)] = d;
        }
    free(img2); free(xy); free(sxs); free(sys);
}

/* L2~ of PAPER.md:160-164 (Monte-Carlo / N-position approximation, used in Eq. 14): the segments are compared with
 * the image only at the start pixels whose mask byte is non-zero; out[i] = number of those starts at which segment
 * vecs[i] lies in phase.  (L2~ = out / N with N = number of selected positions; the caller divides.)  Plain loops. */
void lpf_oracle_counts_masked(const uint8_t *img, const uint8_t *mask, int H, int W, int phase,
                              const int32_t *vecs, int64_t n, int64_t *out)
{
    for (int64_t i = 0; i < n; ++i) {
        int dx = vecs[2 * i], dy = vecs[2 * i + 1];
        int cap = imax_(iabs_(dx), iabs_(dy)) + 1;
        int16_t *xy = (int16_t *)malloc(sizeof(int16_t) * 2 * (size_t)cap);
        int len = lpf_oracle_path(dx, dy, xy);
        int64_t hits = 0;
        for (int y = 0; y < H; ++y)
            for (int x = 0; x < W; ++x) {
                if (!mask[(size_t)y * W + x]) continue;          /* not a selected position */
                int pix;
                for (pix = 0; pix < len; ++pix) {
                    int xx = pmod_(x + xy[2 * pix], W), yy = pmod_(y + xy[2 * pix + 1], H);
                    if (img[(size_t)yy * W + xx] != phase) break;
                }
                if (pix == len) ++hits;
            }
        out[i] = hits;
        free(xy);
    }
}

/* Two-point probability S2 of Eq. 6, un-normalised: for every v = (dx,dy) of the template
 *   out[dy+m][dx+m] = #{ (x1,y1) : chi(x1,y1) = 1 and chi((x1+dx)%W, (y1+dy)%H) = 1 },  chi = [byte == phase];
 * S2 = out / (W*H).  The double sum of Eq. 6 written out; no FFT here (the FFT form, Eq. 7, is a PIN in the tests). */
void lpf_oracle_s2_counts(const uint8_t *img, int H, int W, int phase, int m, int64_t *out)
{
    int S = 2 * m + 1;
    for (int dy = -m; dy <= m; ++dy)
        for (int dx = -m; dx <= m; ++dx) {
            int64_t hits = 0;
            for (int y1 = 0; y1 < H; ++y1)
                for (int x1 = 0; x1 < W; ++x1)
                    if (img[(size_t)y1 * W + x1] == phase &&
                        img[(size_t)pmod_(y1 + dy, H) * W + pmod_(x1 + dx, W)] == phase) ++hits;
            out[(size_t)(dy + m) * S + (dx + m)] = hits;
        }
}

/* Simulated annealing, Alg. 3 with Tab. 2's parameters as arguments, on the integer
 * descriptor.  Readings (the listing is garbled):
 *   A1  one counter n runs over all N proposals (printed: "while c < N_step" although c is reset inside); c and s are
 *       the per-temperature counters, s is incremented on acceptance (missing in the listing)
 *   A2  T_mult = (T_min/T_max)^(s_max/N)  (printed exponent "succ_max/N_step")
 *   A3  the error is minimised: accept iff u < exp((SDP - SDQ)/T) (the printed sign is a maximiser's), evaluated as
 *       ln u < (E_P - E_Q) / ((W*H)^2 * T) with ln u given by the caller: only IEEE * and / are left
 *   A4  SD error = Eq. 19 summed over D (Eq. 13) and over the requested phases, on L = count/(W*H):
 *       e = E/(W*H)^2,  E = sum_phases sum_{v in D} (t_v - c_v)^2  (exact integer)
 *   A5  modify(P) = exchange the bytes of the two pixels of proposal k (given by the caller); a pair
 *       of equal bytes is the identity move (SDQ = SDP: accepted like any other move with no change of error)
 *   phase: 0 | 1 = that phase only, -1 = both (target / counts hold [phase 0][phase 1] then).
 *   use_local = 0: SDQ = evaluate(Q) from scratch, Alg. 3 line 10 literally;  1: counts(Q) = counts(P) + the
 *   local swap delta (pinned to the literal form in the tests; for sizes the literal form cannot reach).
 * img is modified in place; counts_out [n_ph][S][S] = descriptor of the final image (full template, mirrored);
 * stats = { proposals done, accepted, temperature levels finished, final T, final E }; accept_log[N] (may be NULL)
 * gets 1 for every accepted proposal. */
static uint64_t half_sse_(const int64_t *c, const int64_t *t, int m)
{
    int S = 2 * m + 1;
    uint64_t e = 0;
    for (int dy = 0; dy <= m; ++dy)
        for (int dx = -m; dx <= m; ++dx) {
            if (!lpf_oracle_in_half(dx, dy)) continue;
            int64_t d = t[(size_t)(dy + m) * S + (dx + m)] - c[(size_t)(dy + m) * S + (dx + m)];
            e += (uint64_t)(d * d);
        }
    return e;
}

/* Modification operator of Alg. 3 line 9, generated from the CURRENT image ("interchanging two
 * randomly chosen pixels from different phases ... Very simple acceleration employed in our implementation consists in
 * a random selection of interfacial pixels").  The paper does not say how the pixels are drawn; reading A7 of DESIGN.md:
 *   random words: the counter-based generator SplitMix64 (Steele, Lea, Flood 2014; Vigna's splitmix64.c): the n-th
 *     output for `seed` is mix(seed + n * 0x9E3779B97F4A7C15); proposal k, attempt t (0..63), side s (0: p, 1: q) uses
 *     n = 1 + 2 * (64 k + t) + s;  a word u gives the pixel x = ((u >> 32) * W) >> 32, y = ((u & 0xffffffff) * H) >> 32
 *   policy 1 (opposite):    p = attempt 0 of side 0 (any pixel); q = the first attempt of side 1 whose byte differs from p's
 *   policy 2 (interfacial): p = the first attempt of side 0 that is interfacial; q = the first attempt of side 1 that is
 *     interfacial and whose byte differs from p's.  A pixel is interfacial iff one of its 4 periodic neighbours
 *     (x+-1, y), (x, y+-1) has a different byte.
 *   no attempt qualifies (64 tried): q = p, the identity move (reading A5).
 * Rejection from uniform draws = uniform over the qualifying pixels. */
uint64_t lpf_oracle_splitmix64(uint64_t seed, uint64_t n)
{
    uint64_t z = seed + n * 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

static int interfacial_(const uint8_t *img, int H, int W, int x, int y)
{
    uint8_t b = img[(size_t)y * W + x];
    return img[(size_t)y * W + pmod_(x + 1, W)] != b || img[(size_t)y * W + pmod_(x - 1, W)] != b ||
           img[(size_t)pmod_(y + 1, H) * W + x] != b || img[(size_t)pmod_(y - 1, H) * W + x] != b;
}

void lpf_oracle_propose(const uint8_t *img, int H, int W, int policy, uint64_t seed, int64_t k, int32_t *pair)
{
    int px = -1, py = -1, qx = -1, qy = -1;
    for (int t = 0; t < 64 && px < 0; ++t) {
        uint64_t u = lpf_oracle_splitmix64(seed, 1 + 2 * (64 * (uint64_t)k + (uint64_t)t));
        int x = (int)(((u >> 32) * (uint64_t)W) >> 32), y = (int)(((u & 0xffffffffULL) * (uint64_t)H) >> 32);
        if (policy == 1 || interfacial_(img, H, W, x, y)) { px = x; py = y; }
    }
    if (px < 0) {                                   /* no interfacial pixel met: attempt 0 of side 0, identity move */
        uint64_t u = lpf_oracle_splitmix64(seed, 1 + 2 * (64 * (uint64_t)k));
        px = (int)(((u >> 32) * (uint64_t)W) >> 32); py = (int)(((u & 0xffffffffULL) * (uint64_t)H) >> 32);
        pair[0] = px; pair[1] = py; pair[2] = px; pair[3] = py;
        return;
    }
    for (int t = 0; t < 64 && qx < 0; ++t) {
        uint64_t u = lpf_oracle_splitmix64(seed, 1 + 2 * (64 * (uint64_t)k + (uint64_t)t) + 1);
        int x = (int)(((u >> 32) * (uint64_t)W) >> 32), y = (int)(((u & 0xffffffffULL) * (uint64_t)H) >> 32);
        if (img[(size_t)y * W + x] != img[(size_t)py * W + px] && (policy == 1 || interfacial_(img, H, W, x, y))) {
            qx = x; qy = y;
        }
    }
    if (qx < 0) { qx = px; qy = py; }
    pair[0] = px; pair[1] = py; pair[2] = qx; pair[3] = qy;
}

/* policy 0: proposal n is pairs[n] (given); policy 1 | 2: it is generated from the current image by lpf_oracle_propose
 * and written to pairs_out[n] (may be NULL) */
static void anneal_core_(uint8_t *img, int H, int W, int phase, int m, const int64_t *target,
                         const int32_t *pairs, const double *log_u, int64_t N,
                         double T_max, double T_min, int64_t c_max, int64_t s_max, int use_local,
                         int64_t *counts_out, double *stats, uint8_t *accept_log,
                         int policy, uint64_t seed, int32_t *pairs_out)
{
    int S = 2 * m + 1;
    size_t K = (size_t)S * S;
    int n_ph = phase < 0 ? 2 : 1;
    int64_t *cP = counts_out;                                  /* descriptor of P */
    int64_t *cQ = (int64_t *)malloc(sizeof(int64_t) * K * n_ph);
    int32_t *dl = (int32_t *)malloc(sizeof(int32_t) * K);
    for (int i = 0; i < n_ph; ++i)                             /* line 2: SDP = evaluate(P) */
        lpf_oracle_counts(img, H, W, phase < 0 ? i : phase, m, cP + K * i, 0, 0);
    uint64_t EP = 0;
    for (int i = 0; i < n_ph; ++i) EP += half_sse_(cP + K * i, target + K * i, m);
    double T = T_max;                                          /* line 3 */
    double T_mult = pow(T_min / T_max, (double)s_max / (double)N);   /* line 4, reading A2 */
    double wh2 = (double)W * (double)H * (double)W * (double)H;
    int64_t n = 0, accepted = 0, levels = 0;
    while (n < N) {                                            /* line 5, reading A1 */
        int64_t c = 0, s = 0;                                  /* line 6 */
        while (c < c_max && s < s_max && n < N) {              /* line 7 */
            c = c + 1;                                         /* line 8 */
            int32_t gen[4];
            if (policy != 0) {                                 /* line 9: the operator draws its pixels from P */
                lpf_oracle_propose(img, H, W, policy, seed, n, gen);
                if (pairs_out) memcpy(pairs_out + 4 * n, gen, sizeof(gen));
            } else {
                memcpy(gen, pairs + 4 * n, sizeof(gen));
            }
            int xp = gen[0], yp = gen[1], xq = gen[2], yq = gen[3];
            /* line 9: Q = modify(P) */
            uint8_t bp = img[(size_t)yp * W + xp], bq = img[(size_t)yq * W + xq];
            if (use_local) {
                for (int i = 0; i < n_ph; ++i) {
                    lpf_oracle_swap_delta_local(img, H, W, phase < 0 ? i : phase, m, xp, yp, xq, yq, dl);
                    for (size_t k = 0; k < K; ++k) cQ[K * i + k] = cP[K * i + k] + dl[k];
                }
                img[(size_t)yp * W + xp] = bq; img[(size_t)yq * W + xq] = bp;
            } else {
                img[(size_t)yp * W + xp] = bq; img[(size_t)yq * W + xq] = bp;
                for (int i = 0; i < n_ph; ++i)                 /* line 10: SDQ = evaluate(Q) */
                    lpf_oracle_counts(img, H, W, phase < 0 ? i : phase, m, cQ + K * i, 0, 0);
            }
            uint64_t EQ = 0;
            for (int i = 0; i < n_ph; ++i) EQ += half_sse_(cQ + K * i, target + K * i, m);
            double num = (double)((int64_t)EP - (int64_t)EQ);  /* exact: |E| < 2^53 */
            double den = wh2 * T;
            int acc = log_u[n] < num / den;                    /* line 11, reading A3 */
            if (acc) {                                         /* lines 12-13: P = Q, SDP = SDQ */
                memcpy(cP, cQ, sizeof(int64_t) * K * n_ph);
                EP = EQ;
                s = s + 1;
                ++accepted;
            } else {                                           /* undo the modification */
                img[(size_t)yp * W + xp] = bp; img[(size_t)yq * W + xq] = bq;
            }
            if (accept_log) accept_log[n] = (uint8_t)acc;
            ++n;
        }
        if (c >= c_max || s >= s_max) {                        /* the temperature level is complete */
            T = T * T_mult;                                    /* line 17 */
            ++levels;
        }
    }
    stats[0] = (double)n; stats[1] = (double)accepted; stats[2] = (double)levels; stats[3] = T; stats[4] = (double)EP;
    free(cQ); free(dl);
}

void lpf_oracle_anneal(uint8_t *img, int H, int W, int phase, int m, const int64_t *target,
                       const int32_t *pairs, const double *log_u, int64_t N,
                       double T_max, double T_min, int64_t c_max, int64_t s_max, int use_local,
                       int64_t *counts_out, double *stats, uint8_t *accept_log)
{
    anneal_core_(img, H, W, phase, m, target, pairs, log_u, N, T_max, T_min, c_max, s_max, use_local,
                 counts_out, stats, accept_log, 0, 0, NULL);
}

/* Alg. 3 with the modification operator drawing its own pixels (policy 1 | 2 above); pairs_out[N][4] receives the
 * proposal that was decided at every step. */
void lpf_oracle_anneal_generate(uint8_t *img, int H, int W, int phase, int m, const int64_t *target,
                                int policy, uint64_t seed, int32_t *pairs_out, const double *log_u, int64_t N,
                                double T_max, double T_min, int64_t c_max, int64_t s_max, int use_local,
                                int64_t *counts_out, double *stats, uint8_t *accept_log)
{
    anneal_core_(img, H, W, phase, m, target, NULL, log_u, N, T_max, T_min, c_max, s_max, use_local,
                 counts_out, stats, accept_log, policy, seed, pairs_out);
}

int lpf_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
