/* kripke.h - C ABI of the B200-native fused bitmask Kripke evaluator (libkripke_b200.so).
 *
 * What the library computes (citations: P:n = /root/reference/PAPER.md line n):
 *   A batch of modal formulas (postfix programs over T, F, p_i, not, box, dia, and, or, imp;
 *   grammar P:38) is evaluated on every labelled frame of n worlds in a frame class and on every
 *   valuation of n_vars variables, by the bitwise recurrence of P:46-56 (section 3, Lemma 1,
 *   Theorem 1): a world set is an n-bit integer, box x = {w : succ[w] & ~x == 0},
 *   dia x = {w : succ[w] & x != 0}.  Frames and valuations are derived from indices and never
 *   stored (Proposition 1).  Per formula the library returns Algorithm 1's outputs
 *   (P:80-112): the number of refuting (frame, valuation) models, the number of refuting frames,
 *   and the lexicographically first refuting (frame, valuation) with its least falsifying world -
 *   a certificate in the sense of Definition 1.  The pair path returns the same for
 *   "truth sets differ" (Definition 2 / Proposition 4).
 *
 * Index conventions (readings R2, R3):
 *   frame index f:     succ[w] = (f >> (w*n)) & (2^n - 1); bit u of succ[w] is the edge w -> u.
 *   valuation index v: truth(p_i) = (v >> (i*n)) & (2^n - 1); bit w set iff p_i holds at w.
 *   classes:    K all frames; T reflexive; S4 reflexive + transitive; S5 equivalences.
 *   class order:       frames of a class are enumerated by ascending f; a frame range
 *                      [frame_begin, frame_begin + frame_count) indexes that enumeration.
 *   witness.frame is always the K-index f itself.
 *
 * Conventions for every entry point:
 *   - returns KRIPKE_OK (0) or a negative kripke_status; never throws, aborts or prints;
 *   - "host" / "device" on a pointer says where the memory lives; the caller owns every buffer it
 *     passes; the library owns only what a handle holds and frees it in the matching destroy call;
 *   - device work is enqueued on `stream` (a cudaStream_t passed as void*, NULL = default stream)
 *     and the call returns without waiting, unless stated otherwise; outputs are valid once the
 *     stream has been synchronised;
 *   - there is no CPU fallback: without a CUDA device every compute call returns KRIPKE_ECUDA.
 */
#ifndef KRIPKE_H
#define KRIPKE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    KRIPKE_OK = 0,
    KRIPKE_EINVAL = -1,        /* null pointer, size out of range, bad class or flags            */
    KRIPKE_EPROGRAM = -2,      /* malformed postfix program (bad opcode, underflow, != 1 result) */
    KRIPKE_EUNSUPPORTED = -3,  /* valid request outside the implementation limits below         */
    KRIPKE_ECUDA = -4,         /* a CUDA call failed; see kripke_last_cuda_error()               */
    KRIPKE_ENOMEM = -5         /* host allocation failed                                         */
} kripke_status;

/* Postfix opcodes (one byte each).  The paper gives no encoding ("concatenated RPN
 * bytecode"); this one is fixed here.  Binary operators pop y then x and push (x op y). */
enum {
    KRIPKE_OP_TOP = 0x00, KRIPKE_OP_BOT = 0x01,
    KRIPKE_OP_VAR0 = 0x10,                       /* 0x10 + i is variable p_i, i < n_vars <= 4 */
    KRIPKE_OP_NOT = 0x20, KRIPKE_OP_BOX = 0x21, KRIPKE_OP_DIA = 0x22,
    KRIPKE_OP_AND = 0x30, KRIPKE_OP_OR = 0x31, KRIPKE_OP_IMP = 0x32
};

enum { KRIPKE_CLASS_K = 0, KRIPKE_CLASS_T = 1, KRIPKE_CLASS_S4 = 2, KRIPKE_CLASS_S5 = 3 };

/* Implementation limits (the paper's own are P:390: 32-bit masks, 16 successor slots, 48-slot
 * stack, <= 4 variables, k*n < 63). */
#define KRIPKE_MAX_WORLDS 6u
#define KRIPKE_MAX_VARS 4u
#define KRIPKE_MAX_STACK 16u        /* postfix stack slots a program may need               */
#define KRIPKE_MAX_PROGRAM_LEN 64u  /* opcodes per program                                   */
#define KRIPKE_MAX_MODEL_BITS 61u   /* n*n + n_vars*n must not exceed this                   */
#define KRIPKE_LIST_MAX_WORLDS 16u  /* frame-list mode: worlds per explicit frame ("16
                                       successor slots")                                     */
#define KRIPKE_LIST_MAX_VAL_BITS 20u/* frame-list mode: n_vars*n must not exceed this       */

/* flags of the *_range calls */
enum {
    KRIPKE_ACCUMULATE = 1u << 0,      /* add to counts_out / keep the smaller witness instead of
                                         overwriting (chunked scans, multi-GPU shards)            */
    KRIPKE_FULL_SWEEP = 1u << 1,      /* evaluate every program on all 2^(n_vars*n) valuations even if it
                                         ignores a variable (default: a program is scanned over the
                                         valuations of the variables it mentions - the paper's
                                         per-formula k_b, P:93 - and its model count scaled; results
                                         are identical either way)                                 */
    KRIPKE_NO_SHARING = 1u << 2,      /* scan every program itself (default: programs of one call whose
                                         lowered forms are identical - equal after constant folding and
                                         the renaming of the variables they mention - are scanned once
                                         and the others receive the same counts and first refuting
                                         frame; the witness valuation and world are computed per
                                         formula; results are identical either way)                */
    KRIPKE_NO_SUBTERM_SHARING = 1u << 3, /* compiled kernels only: identical programs are still scanned once,
                                         but a subterm that occurs in several programs is evaluated in each
                                         of them (default: the batch is one graph of distinct subterms and
                                         each is evaluated once per 32-model word); ablation                 */
    KRIPKE_KERNEL_AUTO = 0u << 4,     /* compiled bit-sliced kernels where the emitter covers the shape,
                                         else the interpreted bit-sliced kernel, else the scalar one */
    KRIPKE_KERNEL_SCALAR = 1u << 4,   /* force the scalar kernel (Algorithm 1 restated, one model
                                         per thread iteration): baseline / ablation / cross-check */
    KRIPKE_KERNEL_SLICED = 2u << 4,   /* force the interpreted bit-sliced kernel (micro-op dispatch, no
                                         run-time compilation); KRIPKE_EUNSUPPORTED if the shape or a
                                         program does not fit                                      */
    KRIPKE_KERNEL_JIT = 3u << 4,      /* force the compiled bit-sliced kernels (see "Compiled scans"
                                         below); KRIPKE_EUNSUPPORTED if the shape, class or range is
                                         outside what the emitter covers                           */
    KRIPKE_KERNEL_MASK = 3u << 4,
    KRIPKE_REDUCE_BLOCK = 0u << 8,    /* scalar kernel only: one atomic pair per (block, formula),
                                         the paper's revised reduction                     */
    KRIPKE_REDUCE_WARP = 1u << 8,     /* one atomic pair per (warp, formula)                      */
    KRIPKE_REDUCE_THREAD = 2u << 8,   /* one per failing (frame, formula): the paper's original
                                         frame-atomic variant, kept for ablation   */
    KRIPKE_REDUCE_MASK = 3u << 8,
    KRIPKE_NO_GUARDED_ROOTS = 1u << 10, /* compiled kernels only, ablation: test every formula's full truth set (default:
                                         the refutation test is pushed through the conjunctions and boxes at the
                                         top of a formula - box x is refuted by a model iff x fails at a world that
                                         has a predecessor - so those boxes are never evaluated)    */
    KRIPKE_NO_BOX_DISTRIBUTION = 1u << 11 /* compiled kernels only, ablation: evaluate box (x & y) as written (default:
                                         as box x & box y wherever the batch's other formulas make that cheaper)    */
};

/* Outputs, 16 bytes each ("16 bytes per formula"; layout is reading R18). */
typedef struct {
    uint64_t refuting_models;   /* #{(f, v) in range : truth set != all worlds}                  */
    uint64_t refuting_frames;   /* #{f in range : some v refutes}; valid frames = range - this   */
} kripke_count_t;

typedef struct {
    uint64_t frame;             /* K-index f of the first refuting (f, v); UINT64_MAX = none     */
    uint32_t valuation;         /* v                                                             */
    uint32_t world;             /* least w with bit w of the truth set clear (pairs: least w
                                   where the two truth sets differ)                              */
} kripke_witness_t;

#define KRIPKE_NO_WITNESS UINT64_MAX

/* A validated batch of programs, lowered and resident on the current CUDA device. */
typedef struct kripke_programs kripke_programs_t;

const char *kripke_version(void);

/* Last CUDA error code (a cudaError_t) seen by this thread's most recent failing call, 0 if none. */
int kripke_last_cuda_error(void);

/* Checks B = n_formulas postfix programs (HOST pointers): program b is
 * code[offsets[b] .. offsets[b+1]); offsets has B+1 non-decreasing entries.  Each must use only the
 * opcodes above with variable index < n_vars, never underflow, leave exactly one value, be at most
 * KRIPKE_MAX_PROGRAM_LEN long and need at most KRIPKE_MAX_STACK slots.  On success *max_stack_out
 * (optional) is the deepest stack any program needs.  Pure host function, no CUDA. */
int kripke_validate_programs(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                             uint32_t n_vars, uint32_t *max_stack_out);

/* Stages a batch (step H1): validates (as above), lowers each program to the kernels'
 * internal program format and copies both forms to the current device (synchronous; allocates
 * device memory owned by the handle).  code / offsets are HOST pointers and are not retained. */
int kripke_programs_create(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                           uint32_t n_vars, kripke_programs_t **programs_out);
/* Waits until the device has finished the work enqueued on this handle, then frees what it holds.  A handle
 * that only ran scans (kripke_eval_batch*, kripke_distinguish_pairs*, kripke_eval_frames) waits for its own
 * last scan and does not disturb other streams; one that also ran bitmaps, densities, signatures or the size
 * loop waits for the whole device. */
int kripke_programs_destroy(kripke_programs_t *programs);

/* Number of distinct labelled frames in a class (2^(n*n), 2^(n*n-n), preorders, equivalences). */
int kripke_class_size(uint32_t n_worlds, uint32_t frame_class, uint64_t *size_out);

/* Fused corpus scan over one (class, n) layer (Algorithm 1; steps H1-H6): every program
 * of the batch on every frame of the class and every valuation of n_vars variables (n_vars must be
 * the value given at create time).  counts_out / witness_out: DEVICE arrays of n_formulas entries,
 * overwritten. */
int kripke_eval_batch(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                      uint32_t frame_class, kripke_count_t *counts_out,
                      kripke_witness_t *witness_out, void *stream);

/* Same over the class frames [frame_begin, frame_begin + frame_count) only, with `flags`. */
int kripke_eval_batch_range(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                            uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                            uint32_t flags, kripke_count_t *counts_out,
                            kripke_witness_t *witness_out, void *stream);

/* Pairwise distinguishability (step H7): for pair j = (pairs[2j], pairs[2j+1])
 * of program indices, per model x = truth(phi) XOR truth(psi); the model distinguishes the pair
 * iff x != 0; world = least set bit of x.  pairs: HOST array of 2*n_pairs indices (read before the
 * call returns).  counts_out / witness_out: DEVICE arrays of n_pairs entries. */
int kripke_distinguish_pairs(const kripke_programs_t *programs, const uint32_t *pairs,
                             uint32_t n_pairs, uint32_t n_worlds, uint32_t n_vars,
                             uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                             uint32_t flags, kripke_count_t *counts_out,
                             kripke_witness_t *witness_out, void *stream);

/* Size loop and records (step H8; Theorem 2(2)): runs kripke_eval_batch for n = 1..n_max
 * on the full class and keeps, per formula, the least n with a refuting model ("minimal countermodel
 * size", 0 = no countermodel through n_max worlds - never "valid"), the counts of that layer
 * and its first countermodel.  All three outputs are DEVICE arrays of n_formulas entries; enqueued
 * on `stream`. */
int kripke_minimal_refutation(const kripke_programs_t *programs, uint32_t n_vars, uint32_t frame_class,
                              uint32_t n_max, uint32_t *size_out, kripke_count_t *counts_out,
                              kripke_witness_t *witness_out, void *stream);

/* Separation size of formula pairs (Definition 2): for n = 1..n_max scans class K in ascending
 * chunks of at most chunk_frames frames and records, per pair, the least n at which some frame
 * distinguishes it (0 = k-indistinguishable through n_max) and the first distinguishing
 * (frame, valuation, world) of that size.  A pair leaves the scan as soon as it is separated, so
 * the later chunks only carry the survivors.  pairs, size_out, witness_out: HOST arrays
 * (2*n_pairs, n_pairs, n_pairs).  Synchronous. */
int kripke_pairs_separation(const kripke_programs_t *programs, const uint32_t *pairs, uint32_t n_pairs,
                            uint32_t n_vars, uint32_t n_max, uint64_t chunk_frames,
                            uint32_t *size_out, kripke_witness_t *witness_out, void *stream);

/* Frame-list mode (the pairs that survive the exhaustive prefix are "challenged on paths,
 * reverse paths, looped paths, and forked paths of six to ten worlds" / templates "at each size from
 * six through sixteen"; P:192 and Table 2: synthesized relations).  The frames are given, not
 * enumerated: succ is a DEVICE array of n_frames * n_worlds 16-bit successor masks, succ[j*n + w]
 * bit u = edge w -> u of frame j (bits >= n_worlds must be 0), 1 <= n_worlds <= 16,
 * n_vars * n_worlds <= KRIPKE_LIST_MAX_VAL_BITS.  Every program of the batch is evaluated on every
 * listed frame and every valuation; outputs as kripke_eval_batch, with witness.frame =
 * index_base + (position j of the first refuting frame in the list).  flags: KRIPKE_ACCUMULATE
 * (chunked lists: pass each chunk with its index_base), KRIPKE_KERNEL_SCALAR (thread = frame, one
 * model per iteration: cross-check / ablation).  counts_out / witness_out: DEVICE, n_formulas. */
int kripke_eval_frames(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                       const uint16_t *succ, uint64_t n_frames, uint64_t index_base, uint32_t flags,
                       kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream);

/* Frame-list generators (P:183-185 the named stress templates; P:192 / Table 2 the synthesized relations).  The
 * paper's template list and generator parameters are not published; these families take their shape (DESIGN.md
 * 3).  succ_out: DEVICE, n_frames * n_worlds uint16 successor masks in the format above, written on `stream`, so
 * a stress list never exists on the host.  Frame j of a list depends only on (generator, n_worlds, seed, j) and
 * for KRIPKE_GEN_STRESS on n_frames - a counter-based generator, restated in workloads/frames.py for the tests.
 *   KRIPKE_GEN_TEMPLATES    frame j = template j % KRIPKE_TPL_COUNT
 *   KRIPKE_GEN_ERDOS_RENYI  every ordered pair (loops included) is an edge with probability 0.05 / 0.1 / 0.2 /
 *                           0.35 / 0.5 / 0.8 for j % 6 = 0..5 (stratified)
 *   KRIPKE_GEN_EDGE_FLIP    template j % KRIPKE_TPL_COUNT with 1..4 seeded ordered pairs toggled
 *   KRIPKE_GEN_DEAD_END     density-0.3 relation with one seeded world's successors removed
 *   KRIPKE_GEN_BACK_EDGE    the path 0 -> ... -> n-1 plus two seeded edges w -> u, u <= w
 *   KRIPKE_GEN_STRESS       the templates, then the four generators above in equal shares
 * 1 <= n_worlds <= 16, n_frames <= 2^32. */
enum {
    KRIPKE_TPL_PATH = 0, KRIPKE_TPL_REVERSE_PATH = 1, KRIPKE_TPL_REFLEXIVE_PATH = 2, KRIPKE_TPL_FORK = 3,
    KRIPKE_TPL_CYCLE = 4, KRIPKE_TPL_STAR = 5, KRIPKE_TPL_REVERSE_STAR = 6, KRIPKE_TPL_PATH_LOOP_END = 7,
    KRIPKE_TPL_COMPLETE = 8, KRIPKE_TPL_EMPTY = 9, KRIPKE_TPL_COUNT = 10
};
enum {
    KRIPKE_GEN_TEMPLATES = 0, KRIPKE_GEN_ERDOS_RENYI = 1, KRIPKE_GEN_EDGE_FLIP = 2, KRIPKE_GEN_DEAD_END = 3,
    KRIPKE_GEN_BACK_EDGE = 4, KRIPKE_GEN_STRESS = 5, KRIPKE_GEN_COUNT = 6
};
int kripke_frames_generate(uint32_t generator, uint32_t n_worlds, uint64_t n_frames, uint64_t seed,
                           uint16_t *succ_out, void *stream);

/* The pair path over a frame list: pairs is a HOST array of 2*n_pairs program indices;
 * a frame distinguishes pair j under a valuation iff the two truth sets differ; world = least
 * disagreement world.  counts_out / witness_out: DEVICE, n_pairs entries. */
int kripke_distinguish_pairs_frames(const kripke_programs_t *programs, const uint32_t *pairs,
                                    uint32_t n_pairs, uint32_t n_worlds, uint32_t n_vars,
                                    const uint16_t *succ, uint64_t n_frames, uint64_t index_base,
                                    uint32_t flags, kripke_count_t *counts_out,
                                    kripke_witness_t *witness_out, void *stream);

/* Correspondence recovery (Table 9 at P:366-376): "per-formula valid-frame bitmaps ...
 * matched against a first-order condition library".  A bitmap has one bit per class frame of the
 * range [frame_begin, frame_begin + frame_count): bit (j % 32) of word (j / 32) is frame
 * frame_begin + j in class order; words = ceil(frame_count / 32); bits past the range are 0.
 *
 * kripke_validity_bitmap: bit = 1 iff the formula is VALID on the frame (no valuation of the n_vars
 *   variables and no world falsify it).  bitmap_out: DEVICE, n_formulas * words uint32,
 *   formula-major.  (The complement of what refuting_frames counts, per frame.)
 * kripke_condition_bitmap: bit = 1 iff the frame satisfies the first-order condition.  bitmap_out:
 *   DEVICE, words uint32.
 * kripke_match_bitmaps: match_out[r] = least l with bitmaps[r] == library[l] word for word, or
 *   UINT32_MAX.  bitmaps: DEVICE n_records * words; library: DEVICE n_library * words; match_out:
 *   DEVICE n_records. */
enum {
    KRIPKE_COND_REFLEXIVE = 0,            /* T:  box p -> p                                       */
    KRIPKE_COND_TRANSITIVE = 1,           /* 4:  box p -> box box p                               */
    KRIPKE_COND_SYMMETRIC = 2,            /* B:  p -> box dia p                                   */
    KRIPKE_COND_SERIAL = 3,               /* D:  box p -> dia p                                   */
    KRIPKE_COND_EUCLIDEAN = 4,            /* 5:  dia p -> box dia p                               */
    KRIPKE_COND_PARTIALLY_FUNCTIONAL = 5, /* CD: dia p -> box p                                   */
    KRIPKE_COND_DENSE = 6,                /* C4: box box p -> box p                               */
    KRIPKE_COND_CONFLUENT = 7,            /* G:  dia box p -> box dia p                           */
    KRIPKE_COND_COUNT = 8
};
int kripke_validity_bitmap(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                           uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                           uint32_t *bitmap_out, void *stream);
int kripke_condition_bitmap(uint32_t n_worlds, uint32_t condition, uint32_t frame_class,
                            uint64_t frame_begin, uint64_t frame_count, uint32_t *bitmap_out,
                            void *stream);
int kripke_match_bitmaps(const uint32_t *bitmaps, uint32_t n_records, uint64_t words,
                         const uint32_t *library, uint32_t n_library, uint32_t *match_out,
                         void *stream);
/* The frames whose bit is set in a bitmap, written as successor masks in the format of the frame-list
 * calls (so a recovered condition can be re-confirmed on its own extension with kripke_eval_frames:
 * "each re-confirmed over all 33,554,432 five-world frames").  succ_out: DEVICE, capacity *
 * n_worlds uint16; *count_out (DEVICE uint64) = number of set bits; the first min(count, capacity)
 * frames found are written, in unspecified order. */
int kripke_frames_from_bitmap(uint32_t n_worlds, uint32_t frame_class, uint64_t frame_begin,
                              uint64_t frame_count, const uint32_t *bitmap, uint16_t *succ_out,
                              uint64_t capacity, uint64_t *count_out, void *stream);

/* Failure densities - the atlas matrix ("D_ij = the fraction of valuation-world pairs on which
 * formula i fails on ... frame j"; "Atlas-3 concatenates density panels for all frames through
 * three worlds. Atlas-4 and Atlas-5 append stratified panels of 2,048 four-world and 4,096 five-world
 * frames").  counts_out[b * F + j] = #{(v, w) : world w is outside the truth set of formula b under
 * valuation v on frame j}, F = number of frames; D = count / (2^(n_vars*n) * n).  DEVICE uint32,
 * formula-major.  Frames: a class range (n <= 6) or an explicit list of successor masks (n <= 16, the
 * format of kripke_eval_frames).  n_vars * n_worlds <= KRIPKE_LIST_MAX_VAL_BITS. */
int kripke_failure_density(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                           uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                           uint32_t *counts_out, void *stream);
int kripke_failure_density_frames(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                                  const uint16_t *succ, uint64_t n_frames, uint32_t *counts_out,
                                  void *stream);

/* Semantic signatures (the census corpus is "reduced to one representative per semantic equivalence
 * class on all frames of <= 3 worlds"; "64-bit per-size behaviour fingerprint"): sig_out[2b], sig_out[2b+1]
 * = two independent 64-bit sums over every model (frame, valuation) of 1..n_max worlds of a mix of (size, model
 * index, truth set of formula b).  Equal truth sets on all those models give equal signatures; the converse
 * holds up to a ~2^-128 collision, so the hash only screens - a class is made certain with
 * kripke_distinguish_pairs over the same sizes ("no equivalence claim rests on a matching
 * fingerprint").  sig_out: DEVICE, 2 * n_formulas uint64.  1 <= n_max <= 4. */
int kripke_signatures(const kripke_programs_t *programs, uint32_t n_vars, uint32_t n_max, uint64_t *sig_out,
                      void *stream);

/* End-to-end convenience with HOST buffers only: create + eval over the full class + copy the
 * results back + destroy, synchronously (this is what bench.py's "e2e" figure times). */
int kripke_eval_batch_host(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                           uint32_t n_worlds, uint32_t n_vars, uint32_t frame_class,
                           kripke_count_t *counts_host, kripke_witness_t *witness_host);

/* The corpus scan for callers that cannot allocate device memory (Algorithm 1, on the scalar
 * kernel; same results as kripke_eval_batch_range, bit for bit).
 *
 * Why it exists: kripke_programs_create and the scans on a handle call cudaMalloc - for the device copy of
 * the programs, the per-formula accumulators, the S4 / S5 class table, compiled modules.  That rules the
 * handle API out for a process whose device memory is entirely in the hands of another allocator (a torch
 * job whose caching allocator owns the card, a server that reserved its HBM at start-up: cudaMalloc fails
 * there, or takes memory the pool believes is its own), and for a loop that must not stall its other
 * streams (cudaMalloc / cudaFree synchronise the whole device).  This call needs no handle and calls no
 * cudaMalloc, cudaFree or allocating library routine: its working memory - accumulators, the staged
 * programs, the class table - is one fixed block of KRIPKE_STATIC_SCRATCH_BYTES (about 0.8 MB) inside the
 * library image.  Every GPU that loads the library holds that block until the process exits, used or not.
 *
 * Inputs: code / offsets are HOST pointers in the format of kripke_programs_create; they are validated the
 * same way (same status codes) and read before the call returns - unless they lie in page-locked memory,
 * in which case they must stay unchanged until `stream` has passed this call.  Outputs: counts_out /
 * witness_out are the caller's DEVICE arrays of n_formulas entries, written on `stream`.  flags:
 * KRIPKE_ACCUMULATE and KRIPKE_REDUCE_* only (anything else: KRIPKE_EINVAL).
 *
 * Limits, checked on the host before any CUDA call; beyond them the call returns KRIPKE_EUNSUPPORTED and
 * touches nothing: n_formulas <= KRIPKE_STATIC_MAX_FORMULAS; for S4 / S5 the class must have at most
 * KRIPKE_STATIC_MAX_CLASS_FRAMES frames (true for n_worlds <= 5: 6,942 preorders, 52 equivalences).
 *
 * First call on a device: looks up the device address of the block (cudaGetSymbolAddress) with that device
 * current and remembers it; make that first call outside any stream capture.
 *
 * Sharing: all calls on a device use the same block, and it still holds the previous call's contents when
 * the next one starts; each call re-initialises what it reads.  Calls whose device work can overlap -
 * different streams with no event between them, concurrent host threads - race on the block and produce
 * garbage: keep them on one stream or order them with events.
 *
 * Throughput is the scalar kernel's (one model per thread iteration), far below the compiled engine's:
 * this is the escape hatch, not the fast path. */
#define KRIPKE_STATIC_MAX_FORMULAS 8192u
#define KRIPKE_STATIC_MAX_CLASS_FRAMES 8192u
#define KRIPKE_STATIC_SCRATCH_BYTES 819456u
int kripke_eval_batch_static(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                             uint32_t n_worlds, uint32_t n_vars, uint32_t frame_class,
                             uint64_t frame_begin, uint64_t frame_count, uint32_t flags,
                             kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream);

/* What the last eval / pairs call on this handle executed (host-side bookkeeping, valid right
 * after the call returns). */
typedef struct {
    uint32_t launches;                    /* kernel launches enqueued                                  */
    uint32_t kernel_family;               /* which family ran the bulk: 0 scalar, 1 interpreted bit-sliced,
                                             2 compiled bit-sliced                                     */
    uint64_t sliced_logic_ops_per_word;   /* 3-input logic instructions per 32-model word that the scanned
                                             programs need: compiled kernels - what the emitter generated
                                             (each distinct subterm once); interpreted kernel - the lowered
                                             programs' op formula                                        */
    uint64_t models_per_program;          /* definitional: (frames in range) * 2^(n_vars*n)            */
    uint64_t executed_models;             /* models actually evaluated, summed over programs (a program
                                             that mentions g variables is scanned on 2^(g*n) valuations) */
    double logic_instr_per_frame;         /* the same per frame of the range (x words per frame of each
                                             variable-count group): EXECUTED logic thread-instructions   */
    uint32_t jit_programs;                /* distinct programs the compiled kernels evaluated          */
    uint32_t reserved;
    double popc_instr_per_frame;          /* population-count thread-instructions per frame of the range: one per
                                             scanned program and 32-model word (the refuting-model count); they
                                             issue on the quarter-rate XU pipe (16 lanes per clock per SM)       */
    double algorithmic_logic_instr_per_frame; /* SURVEY.md 8(d)'s ALGORITHMIC count: every formula of the
                                             batch as written, no sharing and no folding - (d n^2 + b n +
                                             n + 1) logic instructions per 32-model word (d modal operators,
                                             b binary connectives) x 2^(k_b n) / 32 words per frame, k_b = the
                                             variables the formula mentions.  Work the method defines, not
                                             work the kernels issue                                      */
    double jit_compile_seconds;           /* host time the plan of this call spent in the emitter, NVRTC and
                                             the module load when it was built (0 for interpreted plans)  */
} kripke_run_info_t;
int kripke_last_run_info(const kripke_programs_t *programs, kripke_run_info_t *info_out);

/* Compiled scans.  A batch is known when it is staged, so by default the library turns
 * it into straight-line sm_100a code: all programs of a call become one graph of distinct subterms
 * (negation folded into the operands, or / imp / dia rewritten onto and / box, conjunctions flattened and
 * sorted, variables in a canonical order), groups of at most max_programs_per_kernel programs that share
 * subterms become one kernel each, generated as CUDA C, compiled with NVRTC for sm_100a the first time a
 * (handle, n, class, flags) combination is scanned and cached per process by source text.  That first
 * call therefore blocks for the compilation (kripke_run_info_t.jit_compile_seconds); later calls only
 * enqueue.  Results are identical to the interpreted and scalar kernels (GPU tests).
 * kripke_jit_configure: 1 <= max_programs_per_kernel <= 160 (default 48; more programs per kernel share
 * more subterms and need more registers); 1 <= min_blocks_per_sm <= 8 = the __launch_bounds__ occupancy
 * request of the generated kernels (128 threads per block; default 2, i.e. up to 255 registers per thread).
 * Affects plans built afterwards. */
int kripke_jit_configure(uint32_t max_programs_per_kernel, uint32_t min_blocks_per_sm);

/* Drops everything the process has cached about compiled scans: the plans kept per batch (keyed by the batch's
 * bytes, shape, class and flags) and every loaded module, which is unloaded from the device.  The caches never
 * shrink by themselves - a process that stages corpus after corpus calls this between them to give the host and
 * device memory back - and the next scan of any batch pays the emitter, NVRTC and the module load again (it is
 * also how bench.py measures that cold cost).  Plans cached inside live handles hold kernels of these modules,
 * so the call is refused with KRIPKE_EINVAL while any kripke_programs_t exists; it waits for the device to go
 * idle first (a destroyed handle's last scan may still be running).  *modules_unloaded_out (optional) = number of
 * modules that were loaded. */
int kripke_jit_cache_clear(uint32_t *modules_unloaded_out);

/* Diagnostic (pure host: works without a CUDA device): the CUDA C source of one compiled kernel, exactly as
 * kripke_eval_batch_range / kripke_distinguish_pairs would build it for (n_worlds, frame_class, flags).
 *   batch:        HOST code / offsets as in kripke_programs_create; pairs == NULL for the batch itself, or a
 *                 HOST list of n_pairs pairs of it.
 *   group_vars:   the group of programs that mention this many variables.
 *   kernel_index: which kernel of that group.
 *   compile:      bit 0 = also compile the source with NVRTC to an sm_100a cubin (*cubin_bytes_out);
 *                 bit 1 = the failure-density kernel of kripke_failure_density instead of the scan kernel.
 *   source_out:   capacity cap, NUL-terminated, may be NULL.
 *   *n_kernels_out = kernels of the group; *logic_ops_per_word_out = 3-input logic instructions per 32-model
 *                 word of this kernel.
 * Returns the source length or a negative kripke_status (KRIPKE_EUNSUPPORTED: no compiled layout for the
 * shape). */
int kripke_debug_jit_source(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas, uint32_t n_vars,
                            const uint32_t *pairs, uint32_t n_pairs, uint32_t n_worlds, uint32_t frame_class, uint32_t flags, uint32_t group_vars,
                            uint32_t kernel_index, int compile, char *source_out, uint64_t cap,
                            uint32_t *n_kernels_out, uint64_t *logic_ops_per_word_out, uint64_t *cubin_bytes_out);

/* Diagnostic, host only: for every formula of a batch, whether the model (succ[w] successor masks, val[i] variable
 * masks) refutes it, evaluated on the forms the compiled kernels of (n_worlds, frame_class, flags) evaluate - the
 * batch graph after the guarded-root and box-distribution rewrites, under each record's canonical variable
 * order.  refuted_out: n_formulas bytes (0 / 1).  Returns the number of rewrites applied (>= 0) or an error. */
int kripke_debug_batch_refuted(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas, uint32_t n_vars,
                               uint32_t n_worlds, uint32_t frame_class, uint32_t flags, const uint32_t *succ,
                               const uint32_t *val, uint8_t *refuted_out);

/* Diagnostic (pure host): the truth set (n-bit mask) of one program on one model as the batch graph of the
 * compiled scans computes it - after every rewrite (negation edges, and / box normal form, box
 * distribution, canonical variable order).  succ: n_worlds successor masks; val: n_vars variable masks.
 * Returns the number of graph nodes or a negative kripke_status. */
int kripke_debug_dag_truth(const uint8_t *code, uint32_t len, uint32_t n_vars, uint32_t n_worlds,
                           const uint32_t *succ, const uint32_t *val, uint32_t *truth_out);

/* Integer-pipe calibration ("source-level uint32 XOR/AND/OR" re-done as an instruction
 * rate): runs a register-resident loop of independent 3-input logic instructions on every SM and
 * reports executed thread-instructions per second.  variant: 0 = LOP3 only, 1 = IADD3 only,
 * 2 = SHF only, 3 = LOP3 interleaved with IMAD (reports LOP3+IMAD), 4 / 5 = LOP3 with one / two population
 * counts (each added to a counter with an IMAD) per eight logic instructions - the census loop's own mix; these
 * two report the LOP3 rate alone, so the cost of a POPC shows as the drop against variant 0.  Synchronous. */
int kripke_calibrate_int32(uint32_t variant, double *thread_instr_per_s_out, double *elapsed_ms_out,
                           void *stream);

/* Multi-GPU exchange step: when the frame range of a scan is sharded over
 * ranks, counts combine by SUM and witnesses by lexicographic MIN of (frame, valuation).  These two
 * calls convert DEVICE witness records to and from one 64-bit key per record whose numeric MIN is
 * that lexicographic MIN: key = (((f << n_vars*n) | v) << 3) | world, or 2^63-1 for "none"
 * (n*n + n_vars*n + 3 <= 63 always holds within the limits above), so a single ncclAllReduce(MIN)
 * on the keys and one ncclAllReduce(SUM) on the counts finish the scan. */
int kripke_witness_to_keys(const kripke_witness_t *witness, uint32_t n_records, uint32_t n_worlds,
                           uint32_t n_vars, uint64_t *keys_out, void *stream);
int kripke_keys_to_witness(const uint64_t *keys, uint32_t n_records, uint32_t n_worlds,
                           uint32_t n_vars, kripke_witness_t *witness_out, void *stream);

/* Diagnostic (pure host, no CUDA): lowers one program - or the pair (a, b) if code_b != NULL - to
 * the bit-sliced kernel's 16-bit micro-ops (csrc/ucode.h: low byte op, high byte argument) and
 * copies them to ucode_out (capacity cap entries).  leaf_mode: bit 0 = "box F / dia T is a leaf",
 * bit 1 = "p_0, box p_0, dia p_0 are leaves" (what the kernel instantiation for a shape provides),
 * bit 2 = "fuse a load into the modal operator that follows it".
 * Returns the number of micro-ops, or a negative kripke_status (KRIPKE_EUNSUPPORTED if the program
 * needs more register-stack slots than the kernel has; *need_out is set in both cases). */
int kripke_debug_lower(const uint8_t *code_a, uint32_t len_a, const uint8_t *code_b, uint32_t len_b,
                       uint32_t n_vars, uint32_t leaf_mode, uint16_t *ucode_out, uint32_t cap,
                       uint32_t *need_out);

#ifdef __cplusplus
}
#endif
#endif /* KRIPKE_H */
