/*
 * lpf.h -- C ABI of the B200-native lineal path function library (liblpf.so).
 *
 * What the library computes (Havelka, Kucerova, Sykora, arXiv 1601.04359; citations are
 * PAPER.md lines): for a periodic two-phase pixel image I[y][x] (0<=x<W columns, 0<=y<H
 * rows), a phase phi and every vector v = (dx,dy) of the square template |dx|,|dy| <= m,
 *
 *     count_phi(v) = #{ (x,y) : I[(y+b) mod H][(x+a) mod W] == phi  for all (a,b) in P_v }
 *
 * i.e. the un-normalised lineal path function L2_phi(v) = count_phi(v) / (W*H)
 * (Eq. 8-9; Alg. 1 "for seg / for transl / for pix").
 * P_v is the Bresenham pixel path from (0,0) to v, |P_v| = max(|dx|,|dy|)+1,
 * computed for the canonical half D = {dy>0} u {dy==0, dx>=0} (Eq. 13) with
 * ties rounded up in |minor|, and P_v := reverse(P_{-v}) + v outside D (point symmetry,
 * PAPER.md:140-148).  DESIGN.md "Readings" lists every reading of the paper taken here.
 *
 * Conventions
 *   - Every function returns int: LPF_OK (0) or a negative LPF_E_* code.  Nothing throws,
 *     nothing prints.  lpf_strerror() gives a static string.
 *   - "dev" pointers are CUDA device pointers on the device given to lpf_build_paths;
 *     "host" pointers are ordinary host memory.  All buffers are CALLER-OWNED; the library
 *     owns only what lives inside lpf_paths (the path/trie tables and a packed-image
 *     workspace that grows on demand).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 *     entry points are asynchronous on that stream.  lpf_build_paths and lpf_reserve are the
 *     only calls that allocate device memory, upload tables or synchronise the host: after
 *     lpf_reserve for a shape, lpf_eval / lpf_eval_both / lpf_eval_masked / lpf_eval_sum /
 *     lpf_swap_delta on that shape ONLY enqueue kernels and memsets on `stream` (they can be
 *     captured into a CUDA graph).  A call for a shape that was never reserved reserves it
 *     first, i.e. that one call allocates and synchronises.
 *   - The `const lpf_paths*` of the hot calls: the path table is never modified; the object's
 *     internal caches (plans, workspace, last-launch record) are, so one lpf_paths must not be
 *     used from two host threads at the same time.  Using it from several STREAMS is safe:
 *     consecutive calls share one workspace, so a call on another stream than the previous
 *     call's makes its stream wait, on the device, for the previous call's work.
 *   - There is no CPU fallback: a device entry point called on a table built with
 *     device < 0 returns LPF_E_INVAL.
 */
#ifndef LPF_H_
#define LPF_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LPF_OK             0
#define LPF_E_INVAL       -1   /* null pointer, B<1, phase not in {0,1}, m<0, m > min(H,W)-1, pair out of range */
#define LPF_E_NOMEM       -2   /* host or device allocation failed */
#define LPF_E_CUDA        -3   /* a CUDA runtime call failed (see lpf_last_cuda_error) */
#define LPF_E_UNSUPPORTED -4   /* shape outside what the kernels take (m > 511, one row band + halo > shared memory) */
#define LPF_E_TOO_LARGE   -5   /* lpf_swap_delta_static: the image needs more than LPF_STATIC_SCRATCH_BYTES of scratch */

/* flags of lpf_eval / lpf_eval_both */
#define LPF_PRUNE    1u   /* paper's "enhanced" variant: skip a sub-trie whose running
                             mask is all-zero for the whole block.  Exact: never changes a count. */
#define LPF_NO_TRIE  2u   /* one chain per path P_v (no prefix sharing): the "one-path-per-warp" design
                             variant, kept for the measurement in DESIGN.md. Same counts. */

#define LPF_S2       4u   /* two-point probability instead of the lineal path: only the two END pixels of every
                             segment are tested, counts[v] = #{x : I[x] and I[x+v] in phase} = W*H*S2(v), Eq. 6
                             (PAPER.md:99); same kernels, a program of 2-pixel "paths".  Exact integers (the paper's
                             FFT form, Eq. 7, is floating point). */

#define LPF_NO_E2    8u   /* measurement: walk every node on the plain bit plane instead of the eroded planes (one
                             plane per K-step pattern of a path, K + 1 pixels per window).
                             Same counts. */

#define LPF_LAYOUT_MAX_CLASSES 128
#define LPF_LAYOUT_INTS (10 + 41 * LPF_LAYOUT_MAX_CLASSES)   /* lpf_paths_program */

/* `what` of lpf_reserve */
#define LPF_FOR_EVAL        1u   /* lpf_eval and one-phase lpf_eval_sum with (B, H, W, flags) */
#define LPF_FOR_EVAL_BOTH   2u   /* lpf_eval_both and two-phase lpf_eval_sum */
#define LPF_FOR_MASKED      4u   /* together with one of the above: lpf_eval_masked (one phase / both) instead */
#define LPF_FOR_SWAP_DELTA  8u   /* lpf_swap_delta on H x W images (B, flags unused) */
#define LPF_FOR_ANNEAL     16u   /* lpf_anneal on H x W images (B, flags unused) */
#define LPF_FOR_HOST       32u   /* lpf_eval_host with (B, H, W, flags), one phase or both */

typedef struct lpf_paths lpf_paths;   /* opaque: path table + prefix trie + device programs for one m */

const char* lpf_strerror(int code);
/* Last CUDA error code (cudaError_t as int) recorded by a call that returned LPF_E_CUDA. */
int lpf_last_cuda_error(void);

/* Paper "step 1": rasterise P_v for every v in D with |dx|,|dy| <= m,
 * build the prefix trie over the ordered pixel lists, and keep it (host) for program
 * generation.  device >= 0: also binds the object to that CUDA device; device < 0: host-only
 * table (lpf_paths_info / lpf_paths_get / lpf_paths_program work; device entry points refuse).
 * Errors: m < 0 -> INVAL; m > 511 -> UNSUPPORTED; NOMEM; CUDA. Synchronous. */
int  lpf_build_paths(int m, int device, lpf_paths** out);
void lpf_free_paths(lpf_paths* p);

/* Sizes of the table: |D| = 2m^2+2m+1, sum_v |P_v| (= Eq. 17 with W = m+1,
 * PAPER.md:186-196), number of trie nodes (distinct path prefixes, root included), and the
 * deepest node (= m). Any out pointer may be NULL. */
int  lpf_paths_info(const lpf_paths* p, int64_t* n_half_vectors, int64_t* sum_path_len,
                    int64_t* n_trie_nodes, int* max_depth);

/* Host: P_v for ANY v of the template (|dx|,|dy| <= m).  xy = host [cap][2] int16 (x then y),
 * *len = |P_v|; INVAL if v is outside the template or cap < |P_v|. */
int  lpf_paths_get(const lpf_paths* p, int dx, int dy, int16_t* xy, int cap, int* len);

/* Host, for tests and tools: the linearised walk program the eval kernel interprets for H x W images
 * (DESIGN.md "Node program").  Every v in D is walked in one of four octant VIEWS of the image (transposed /
 * flipped so that the path is x-major with a' >= 0, 0 <= b' <= a'); each octant has its own prefix trie, cut
 * into connected pieces of about `piece_nodes` nodes (<= 0: one piece per octant); each piece is one item =
 * the chain from the root to the piece root followed by the piece in depth-first order.  flags: 0, LPF_NO_TRIE, LPF_S2, LPF_NO_E2.
 *   entries  host [cap_entries] uint64 (may be NULL to query sizes); low word: bits 0-4 a' & 31, bit 5 reload,
 *            6 terminal, 7 save, 8 restore, 9 init, 10 pair (own mask never needed, the next entry continues from it),
 *            bits 12-31 b' * stride + (a' >> 5) (+ q * band_words); high word: bits 0-19
 *            (dy+m)*(2m+1) + (dx+m) in IMAGE coordinates, 20-22 restore slot, 23-25 save slot, 26-28 q, 29-30 back.
 *            bit 11: the window is read from an eroded plane (program of level K >= 1: every entry).  The plane of
 *            step pattern q holds, at (a', b'), the AND of the K + 1 pixels (a' + j, b' + s_1 + .. + s_j), j = 0..K,
 *            s_j = bit j-1 of q -- K + 1 consecutive pixels of a first-octant path.  Some first pixels of the window may
 *            be nodes that are already in the mask; the others are the nodes of this entry; terminal / save / count
 *            index are the last one's.  The vectors of an octant are split by slope into pattern CLASSES whose paths use
 *            few patterns; an item belongs to one class and its entries address the class's planes by slot:
 *            bits 12-31 = b' * stride + (a' >> 5) + slot * (band words of the class); high word bits 26-31 repeat q.
 *            At level K no window ends above depth K: every item starts (its first and only init entry) with the
 *            window root .. depth K, and the vectors shorter than that are counted by a separate small kernel.
 *   items    host [cap_items][4] int64 = (first entry, number of entries, octant, pattern class) (may be NULL)
 *   layout   host int[LPF_LAYOUT_INTS]: [0..3] words per packed row of each octant view (decodes b', a' >> 5), [4..7]
 *            words of one full-height band of each view (0 for the plain program), [8] the level K of the program
 *            (0: plain), [9] the number of pattern classes, then per class 41 ints: octant, patterns used n, words of one
 *            band of THIS class in shared memory (the plane in slot s sits at s times that; a class keeps only the rows
 *            its paths reach), rows of that band, the level of the class (the K of ITS windows: the program's, or lower
 *            for steep slopes of a template that is large against the image), the pattern q of slot 0 .. n-1 (-1 beyond)
 * *n_entries / *n_items / *n_slots (mask-stack slots the program needs) are always written.
 * Octants (view coordinates a', b' from image coordinates a, b): 0: dx>=0, dy<=dx (a,b); 1: dx>=0, dy>dx (b,a);
 * 2: dx<0, dy>-dx (b,-a); 3: dx<0, dy<=-dx (-a,b). */
int  lpf_paths_program(lpf_paths* p, int H, int W, int piece_nodes, unsigned flags,
                       uint64_t* entries, int64_t cap_entries, int64_t* n_entries,
                       int64_t* items, int64_t cap_items, int64_t* n_items, int* n_slots, int* layout);

/* The rest of paper "step 1" for one image shape (step 1 is executed once, steps 2-3 "are called
 * repeatedly ... for new binary images of the same dimensions"): cuts the tries into the work items of a B x H x W
 * batch, linearises and uploads the node program, sizes every device workspace the named calls need and fixes their
 * launch configuration.  `what` is an OR of LPF_FOR_*; `flags` are the eval flags the later calls will pass.
 * Synchronous (allocates, copies, synchronises the device).  After it the named calls on that shape only enqueue work
 * on their stream.  May be called any number of times; a larger shape grows the workspace (the device is synchronised
 * first, so work in flight is safe).  Errors: INVAL, UNSUPPORTED, NOMEM, CUDA as for the calls themselves. */
int  lpf_reserve(lpf_paths* p, int B, int H, int W, unsigned flags, unsigned what);

/* Paper "steps 2-3" (Alg. 1 / Alg. 2) for a batch of B independent images
 * of one size: translate every segment over every start pixel, compare, count.
 *   images  dev uint8 [B][H][W]; a pixel is in phase phi iff its byte == phi
 *   counts  dev int64 [B][2m+1][2m+1], index [b][dy+m][dx+m]; fully overwritten
 *           (the half outside D is the mirror counts[-v] = counts[v])
 * Errors: INVAL (see above; m > min(H,W)-1 is rejected because a path would wrap onto itself,
 * and D stops at W-1,H-1: PAPER.md:154), UNSUPPORTED, NOMEM, CUDA. */
int  lpf_eval(const lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase,
              int64_t* counts, unsigned flags, void* stream);

/* Monte-Carlo / N-position approximation L2~ (used in Eq. 14): the segments are compared with the
 * image only at the selected start positions.
 *   start_mask dev uint8 [H][W], shared by the whole batch: a start pixel is selected iff its byte is non-zero
 *   phase      0 | 1: counts dev int64 [B][2m+1][2m+1];  -1: both phases, counts dev int64 [B][2][2m+1][2m+1]
 * counts[v] for v in D (Eq. 13) = number of selected starts at which P_v lies in phase (L2~ = counts / N, the caller
 * divides by its N); the half outside D repeats it point-symmetrically, as the descriptor is stored in the paper
 * -- with a proper subset of starts the definition itself is not symmetric (reading S16).
 * A mask of all non-zero bytes gives exactly lpf_eval.  Same errors as lpf_eval. */
int  lpf_eval_masked(const lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase,
                     const uint8_t* start_mask, int64_t* counts, unsigned flags, void* stream);

/* Both phases in one call: counts dev int64 [B][2][2m+1][2m+1], index [b][phase][dy+m][dx+m]. */
int  lpf_eval_both(const lpf_paths* p, const uint8_t* images, int B, int H, int W,
                   int64_t* counts, unsigned flags, void* stream);

/* Ensemble descriptor of an image stack (the descriptor of the bone specimen is "averaged over 100
 * slices", ergodicity): counts_sum[v] = sum over the B images of count(image_b, v), accumulated on the device into ONE
 * array without materialising the per-image counts; the ensemble average of L2 is counts_sum / (B*W*H), one division
 * done by the caller.  With LPF_S2 the same for the two-point probability.
 *   phase 0 | 1: counts_sum dev int64 [2m+1][2m+1];  -1: both phases, dev int64 [2][2m+1][2m+1].
 * Same errors as lpf_eval. */
int  lpf_eval_sum(const lpf_paths* p, const uint8_t* images, int B, int H, int W, int phase,
                  int64_t* counts_sum, unsigned flags, void* stream);

/* Least-square objective, Eq. 14 / Eq. 19 on integer counts:
 *   sse[b] = sum_k (counts[b][k] - target[k])^2, exact in uint64 (wraps mod 2^64 if it overflows;
 *   it cannot for counts <= 2^26 and K <= 2^12 ... see DESIGN.md).  e = sse / (W*H)^2 is the caller's.
 *   counts dev int64 [B][K], target dev int64 [K], sse dev uint64 [B]. */
int  lpf_objective(const int64_t* counts, const int64_t* target, int B, int64_t K,
                   uint64_t* sse, void* stream);

/* Two-pixel swap: for each of n INDEPENDENT proposals against one base
 * image, delta[i][dy+m][dx+m] = count_phase(I_i', v) - count_phase(I, v), where I_i' is I with
 * the bytes of pixels p_i and q_i exchanged.  Only segments through p or q are re-tested.
 *   image dev uint8 [H][W]; pairs dev int32 [n][4] = x_p, y_p, x_q, y_q; delta dev int32 [n][2m+1][2m+1].
 * Pairs are range-checked on the device; an out-of-range pair yields an all-zero delta and the
 * call still returns LPF_OK (no host sync) -- validate on the host if needed.
 * UNSUPPORTED when the bit image with its halo of m pixels, (H+2m) x ceil((W+2m)/32) words, plus 32 KB of warp stacks
 * does not fit the shared memory of one block, or when the trie has 2^24 nodes or more (m > ~380). */
int  lpf_swap_delta(const lpf_paths* p, const uint8_t* image, int H, int W, int phase,
                    const int32_t* pairs, int64_t n, int32_t* delta, void* stream);

/* lpf_swap_delta for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): same arguments, same result, but the scratch of the evaluation (the bit images of
 * the phase and their copy with a halo of m pixels) lives in ONE array of LPF_STATIC_SCRATCH_BYTES in the library's
 * device image, which every GPU that loads the library holds until the process exits.  The call never calls
 * cudaMalloc, cudaFree or an allocating library routine: it enqueues memsets and kernels on `stream` and returns.
 *   - The node records of the trie belong to p and are uploaded by lpf_reserve(p, 1, H, W, 0, LPF_FOR_SWAP_DELTA)
 *     (any H, W: they do not depend on the shape) or by an earlier lpf_swap_delta: LPF_E_INVAL if neither happened.
 *   - LPF_E_TOO_LARGE if 4 * (H*ceil(W/32) + W*ceil(H/32) + (H+2m)*ceil((W+2m)/32)) + 256 bytes exceed
 *     LPF_STATIC_SCRATCH_BYTES = 256 KiB (config 5, 256 x 256 with m = 64, needs 35 KB; 768 x 768 with m = 32 fits,
 *     1024 x 1024 does not).  Otherwise the errors of lpf_swap_delta.
 *   - All calls on one GPU share the array, whatever their lpf_paths or stream: calls that overlap on the GPU race;
 *     order them (one stream, or events).  The array keeps the last call's contents; every call clears what it reads.
 *   - The first call on a device looks up the array's device address (cudaGetSymbolAddress; the runtime may load the
 *     library's device image then): make it before a graph capture begins. */
#define LPF_STATIC_SCRATCH_BYTES (256 * 1024)
int  lpf_swap_delta_static(const lpf_paths* p, const uint8_t* image, int H, int W, int phase,
                           const int32_t* pairs, int64_t n, int32_t* delta, void* stream);

/* Simulated annealing of Alg. 3 with the two-pixel swap and the least-square
 * error of Eq. 19 on the lineal path descriptor; Tab. 2's parameters are arguments.  Readings A1-A5 of
 * the garbled listing are listed in DESIGN.md "Annealing readings".  The chain is exactly the sequential one:
 * proposal k exchanges the bytes of pixels (x_p,y_p), (x_q,y_q) = pairs[k]; it is accepted iff
 * log_u[k] < (E_P - E_Q) / ((W*H)^2 * T), E = sum over the phases and v in D of (target - counts)^2; a pair of equal
 * bytes (or out of range) is the identity move; T *= (T_min/T_max)^(s_max/N) whenever c_max proposals or s_max
 * acceptances were seen at the current temperature.  Batches of consecutive proposals are evaluated speculatively in
 * parallel (the swap-delta evaluation) and decided in order on the device; the whole chain is ONE cooperative kernel
 * launch (workspace: lpf_reserve with LPF_FOR_ANNEAL).
 *   image dev uint8 [H][W], modified in place      phase 0 | 1 | -1 (both: target/counts are [2][2m+1][2m+1])
 *   target dev int64 [n_ph][2m+1][2m+1]            pairs dev int32 [N][4], log_u dev double [N] (ln of uniforms in [0,1))
 *   counts dev int64 [n_ph][2m+1][2m+1]: descriptor of the final image      accept_log dev uint8 [N] or NULL
 *   stats5 HOST double[5] = { proposals done, accepted, temperature levels completed, final T, final E }
 * Synchronous: returns when the chain is finished.  Errors as lpf_eval / lpf_swap_delta. */
int  lpf_anneal(lpf_paths* p, uint8_t* image, int H, int W, int phase, const int64_t* target, const int32_t* pairs,
                const double* log_u, int64_t N, double T_max, double T_min, int64_t c_max, int64_t s_max,
                int64_t* counts, uint8_t* accept_log, double* stats5, void* stream);

/* lpf_anneal with the modification operator drawing its own pixels from the current image ("two
 * randomly chosen pixels from different phases"; "a random selection of interfacial pixels", the acceleration the paper
 * uses).  The paper does not say how they are drawn; reading A7: proposal k, attempt t = 0..63, side s (0: p,
 * 1: q) uses output n = 1 + 2 (64 k + t) + s of SplitMix64 seeded with `seed`; a word u gives the pixel
 * x = ((u >> 32) * W) >> 32, y = ((u & 0xffffffff) * H) >> 32.
 *   LPF_PROPOSE_OPPOSITE:    p = attempt 0 of side 0; q = the first attempt of side 1 whose byte differs from p's
 *   LPF_PROPOSE_INTERFACIAL: p = the first interfacial attempt of side 0; q = the first interfacial attempt of side 1
 *                            whose byte differs from p's (interfacial: one of the 4 periodic neighbours has another byte)
 *   nothing qualifies: q = p, the identity move.
 *   pairs_out dev int32 [N][4]: the proposal decided at every step (written by the device; required)
 * Everything else as lpf_anneal (log_u stays an input: the logarithm is not bit-reproducible across libraries). */
#define LPF_PROPOSE_OPPOSITE    1
#define LPF_PROPOSE_INTERFACIAL 2
int  lpf_anneal_generate(lpf_paths* p, uint8_t* image, int H, int W, int phase, const int64_t* target, int policy,
                         uint64_t seed, int32_t* pairs_out, const double* log_u, int64_t N, double T_max, double T_min,
                         int64_t c_max, int64_t s_max, int64_t* counts, uint8_t* accept_log, double* stats5,
                         void* stream);

/* HOST-buffer convenience used by the end-to-end measurement: copies `images` (host, pinned or
 * not) to the device on a private stream (ordered after earlier work on this table), runs lpf_eval (_both if
 * phase < 0), copies counts back, synchronises that stream.  Staging buffers: lpf_reserve with LPF_FOR_HOST. */
int  lpf_eval_host(lpf_paths* p, const uint8_t* images_host, int B, int H, int W, int phase,
                   int64_t* counts_host, unsigned flags);

/* Counters of the most recent lpf_eval / lpf_eval_both on this object (host values known at
 * launch time): kernels launched, work units x (image group, phase), program entries walked per
 * image-phase, grid, block, dynamic shared memory bytes, thread tile code (1000 TX + 100 TY + 10 if the mask stack is in
 * tensor memory + mask-stack slots), images
 * per team, the erosion level K of the program (0: the plain plane); then what the walker executes per image-phase and
 * per start WORD, counted by replaying its loop over the program on the host: pairs of entries folded into one
 * 3-input AND (2 SHF + 1 LOP3 each), entries executed on their own (1 SHF + 1 LOP3), terminal entries (1 POPC +
 * 1 add), the trie nodes per program piece; the teams per CTA, the CTAs resident per SM, the vectors shorter than K
 * that the small extra kernel counts, the entries that reload their row strip from shared memory (TY * (TX + 1) 32-bit
 * loads per thread each) and the number of pattern classes.  out = host int64[18]. */
int  lpf_last_launch_info(const lpf_paths* p, int64_t* out18);

/* Measurement hook: with enable != 0 every lpf_eval / lpf_eval_both on this object
 * records one CUDA event before and one after the eval kernel (the dominant kernel) on the caller's
 * stream; lpf_last_eval_kernel_ms waits for the second event and returns the elapsed device time of
 * the most recent eval kernel in milliseconds.  INVAL if no timed eval has been issued. */
int  lpf_set_timing(lpf_paths* p, int enable);
int  lpf_last_eval_kernel_ms(const lpf_paths* p, float* ms);

/* Measurement hook: runs a few milliseconds of register-only
 * integer instructions on every SM of `device` (synchronous, default stream) and returns the measured thread-level
 * instruction rates in ops/s: out4 = { LOP3, SHF.R.W, the eval kernel's SHF+SHF+LOP3 pair pattern, POPC }.
 * It is the measured counterpart of the derived peak bench.py reports against; it touches no lpf_paths state. */
int  lpf_alu_peak(int device, double* out4);

/* Tuning hook: overrides the thread tile of the eval kernel -- TX x-adjacent words x
 * TY start rows per thread, (TX,TY) in {(4,2),(8,1),(4,4),(8,2),(16,1)}, and the warps per CTA (1..8) -- for the
 * following lpf_eval calls on this object; 0 = automatic choice.  Never changes a count.  INVAL otherwise. */
int  lpf_set_tile(lpf_paths* p, int tx, int ty, int cta_warps);

/* Tuning hook: caps the erosion level of the programs built for the following
 * lpf_reserve / lpf_eval / lpf_paths_program calls on this object: 0..6, or -1 = automatic (the default).  Level K
 * keeps the planes of one pattern class per row band in shared memory; the highest level that fits and keeps enough
 * warps resident is the fastest.  Where a template is large against the image, the classes of steep slopes run below
 * the program's level (the level of each class is in the layout of lpf_paths_program).  LPF_NO_E2 is level 0.  Never
 * changes a count.  INVAL otherwise. */
int  lpf_set_level(lpf_paths* p, int max_level);

/* Tuning hook: the dynamic shared memory one CTA of the eval kernel may use, in bytes, for
 * the following lpf_reserve / lpf_eval / lpf_paths_program calls on this object: >= 16384, or 0 = all the device gives
 * (the default; more than the device gives is the same).  With less room fewer planes fit beside a band: the bands get
 * lower, then the pattern classes of steep slopes run at lower levels than the program's (as they do for templates
 * that are large against the image), then the level drops.  Never changes a count.  INVAL otherwise. */
int  lpf_set_shared_memory(lpf_paths* p, int bytes);

/* Tuning hook: where the walker keeps the masks it saves at the branching nodes
 * of the trie.  enable = 1 (the default): in TENSOR MEMORY (tcgen05.st / tcgen05.ld) whenever the launch runs one CTA
 * per SM and the slots of all its warps fit the 512 columns -- the big shapes; 0: always in local memory, as the small
 * shapes do.  For the following lpf_reserve / lpf_eval calls on this object.  Never changes a count.  INVAL otherwise. */
int  lpf_set_tmem_stack(lpf_paths* p, int enable);

/* Tuning hook: a CTA of the eval kernel is n_teams teams that share the row bands it holds in
 * shared memory; every team walks its own work unit (the segments are distributed, the image is shared).
 * n_teams = 1..32 fixes the number for the following lpf_reserve / lpf_eval calls on this object (shapes whose CTA would
 * exceed 1024 threads are refused, LPF_E_UNSUPPORTED), 0 = automatic (the count that keeps the most warps resident).
 * Never changes a count.  INVAL otherwise. */
int  lpf_set_teams(lpf_paths* p, int n_teams);

#ifdef __cplusplus
}
#endif
#endif /* LPF_H_ */
