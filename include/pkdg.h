/*
 * pkdg.h -- C ABI of pkdg-b200: per-bucket evaluation of gravity interaction lists on one
 * NVIDIA B200 (sm_100a), after PKDGRAV3 (Potter, Stadel & Teyssier, arXiv 1609.08621).
 *
 * Problem statement: leaf cells ("buckets") hold up to
 * b ~ 16 sink particles; the tree walk gives every sink a P-P list of source particles and a
 * P-C list of source cells whose multipole moments (to 4th order, about the cell's centre of
 * mass) stand for their mass; evaluating the lists gives the acceleration and the potential of
 * every sink particle.  The paper runs exactly this on the GPU (sec 3.3).  The formulas are not
 * printed in the paper; DESIGN.md (readings A1-A18) fixes them:
 *
 *   P-P: d = x_i - x_j, h = 2 eps, u = |d|/h; a_i -= m_j d g(u)/h^3, phi_i += m_j w(u)/h, with
 *        g, w of the cubic-spline softened pair (exactly Newtonian for |d| >= 2 eps).  A source
 *        whose INDEX equals the sink's index is skipped; distinct coincident particles interact.
 *   P-C: r = x_i - COM_c; phi_i += - sum_{|k| in {0,2,3,4}} (-1)^|k| M_k t_k(r), a_i = -grad of
 *        that truncated potential, t_k = d^k(1/|r|)/k!; unsoftened; dipole dropped.
 *
 * Conventions.  G = 1.  Every pointer is a DEVICE pointer unless its name ends in _host.  The
 * caller owns every buffer; the library never frees, reallocates or retains caller memory after
 * the work queued by a call has completed.  Calls are asynchronous on `stream` (a cudaStream_t
 * passed as void*; NULL = the legacy default stream) unless stated; no exception crosses the
 * ABI; every function returns a pkdg_status (0 = OK, < 0 = error) and pkdg_last_error() gives
 * the text.  A pkdg_ctx may be used by one host thread at a time.
 *
 * Precision ("single precision in calculating interactions, but all components are
 * accumulated in double precision").  Terms and per-lane
 * partial sums are fp32.  Beside a_i the kernel accumulates S2_i = sum_j |a_ij|^2; a sink whose sum cancels
 * so far that fp32 terms cannot give 2e-5 of |a_i| (sqrt(S2_i) > kappa2 |a_i|, default kappa2 = 6, option
 * PKDG_OPT_KAPPA2) is re-evaluated over the same lists by a second kernel with fp64 terms and fp64
 * accumulators and its row is written by that kernel.  pkdg_stats.fixup_sinks counts them.
 *
 * Stream order.  Consecutive calls on ONE context must be stream-ordered (same stream, or ordered by
 * events): they share the context's workspace (descriptors, counters, queues).  eps == 0: pairs closer
 * than 1e-12 are treated as coincident and contribute nothing (the Newtonian pair is undefined there).
 *
 * Value range.  Coordinates must satisfy |x| <= 1e12 and masses must be finite: the kernels park
 * masked list entries (padding, out-of-range indices) at +1e15 with mass 0 and unused sink slots at
 * -1e15, and rely on those never coming within fp32 range of a real particle.  Cell records must
 * have b_max / |x_sink - COM| < 1 for every listed pair (any sensible opening criterion does).  The
 * flag PKDG_VALIDATE checks all of this on the device.
 */
#ifndef PKDG_H
#define PKDG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PKDG_VERSION_MAJOR 0
#define PKDG_VERSION_MINOR 2

#define PKDG_TILE 32          /* list entries per tile = lanes per warp */
#define PKDG_CELL_FLOATS 36   /* canonical cell record, see pkdg_cells */
#define PKDG_PAD (-1)         /* index that pads the last tile of a list */

typedef int32_t pkdg_status;
#define PKDG_OK 0
#define PKDG_EINVAL (-1)   /* null pointer, negative size, bad stride, misaligned buffer */
#define PKDG_ECUDA (-2)    /* a CUDA runtime call failed; text in pkdg_last_error() */
#define PKDG_ENOMEM (-3)   /* workspace allocation failed */
#define PKDG_EBADLIST (-4) /* validation found a non-monotone offset, an index out of range or a
                              negative bucket count (only reported by pkdg_get_stats) */
#define PKDG_EBADVALUE (-5) /* PKDG_VALIDATE found values or geometry outside the documented range
                               (only reported by pkdg_get_stats) */

/* flags of pkdg_gravity_eval* */
#define PKDG_ACCUMULATE 0x1u /* add to out instead of overwriting it */
#define PKDG_SKIP_PP 0x2u    /* ignore the P-P lists (kernel studies) */
#define PKDG_SKIP_PC 0x4u    /* ignore the P-C lists */
#define PKDG_PP_LEAVES 0x8u  /* the P-P list's entries are BUCKET indices (into `buckets`), each standing for
                                all particles of that bucket, <= 16 of them (SURVEY.md sec 8(f) NEXT-1,
                                range-compressed P-P entries; a leaf that fails the
                                opening test joins the P-P list whole).  16 times fewer list bytes and
                                contiguous source gathers.  interactions_pp counts the particles the
                                references stand for, tiles_pp two references per tile.  With the
                                streamed variants `buckets_host` must hold ALL buckets a reference may
                                name (it always does: references index it).                           */
#define PKDG_VALIDATE 0x40u  /* check the value-range contract below on the device (two extra kernels): every
                                coordinate finite and |x| <= 1e12, masses and moments finite
                                (invalid_values), every listed (sink, cell) pair with the sink outside the
                                cell's b_max sphere (invalid_pairs); reported by pkdg_get_stats          */
#define PKDG_NO_FIXUP 0x10u  /* do not re-evaluate ill-conditioned sinks in fp64 (see "Precision" below)   */
#define PKDG_FIXUP_ALL 0x20u /* send EVERY sink through the fp64 fix-up kernel (fp64 terms and fp64
                                accumulators throughout: the cost of PAPER.md:L83's double-precision
                                accumulation, measured by bench.py --report; also the test of that kernel) */

typedef struct pkdg_ctx pkdg_ctx;

/* Sink and source particles, tree order (buckets are contiguous runs).  xyzm = [n][4] fp32
 * (x, y, z, mass), 16-byte aligned.  ("hierarchically sorted order"; L83 fp32.) */
typedef struct { const float *xyzm; int64_t n; } pkdg_particles;

/* Source cells.  rec = [n][stride_floats] fp32, stride_floats >= 36.  Canonical record:
 * [0..2] centre of mass (the centre of expansion), [3] mass, [4..9] 2nd, [10..19]
 * 3rd, [20..34] 4th raw moments M_k = sum_j m_j s_x^a s_y^b s_z^c about that centre, for each
 * order n in the sequence a = n..0, b = n-a..0, c = n-a-b (n = 2: xx xy xz yy yz zz), [35] b_max,
 * the distance from the centre to the farthest particle (used only as the length
 * scale of the internal normalised form; <= 0 means "derive a scale from the 2nd moments"). */
typedef struct { const float *rec; int64_t n; int32_t stride_floats; } pkdg_cells;

/* Buckets: sinks first[b] .. first[b]+count[b]-1.  count >= 0 (tuned for <= 16).
 * Buckets must not overlap unless PKDG_ACCUMULATE semantics are not needed. */
typedef struct { const int32_t *first; const int32_t *count; int64_t n; } pkdg_buckets;

/* A CSR interaction list: entries offsets[b] .. offsets[b+1]-1 of idx belong to bucket b
 * (offsets has n_buckets+1 int64 values, offsets[0] may be non-zero).  idx < 0 is padding and
 * is ignored.  A NULL pkdg_list* or NULL offsets means "no list of this kind". */
typedef struct { const int64_t *offsets; const int32_t *idx; } pkdg_list;

/* Groups of consecutive buckets that SHARE one P-P and one P-C list (PAPER.md:L69:
 * "If a source cell is reached with fewer than g particles (called the group size) we proceed no deeper in
 * the tree resolving the remaining checklist into interaction lists ... a group size of 64, or more
 * generally four times the bucket size").  Group g holds buckets first_bucket[g] .. first_bucket[g] +
 * n_buckets[g] - 1; the groups must tile the bucket range in order.  With groups the lists have n + 1
 * offsets (one list per group) and every sink of the group's buckets evaluates the whole list. */
typedef struct { const int32_t *first_bucket; const int32_t *n_buckets; int64_t n; } pkdg_groups;

/* Counters of the last evaluation on a context (pkdg_get_stats synchronises the stream). */
typedef struct {
    int64_t n_buckets;
    int64_t interactions_pp; /* I_pp = sum_b count[b] * len_pp[b]  (padding entries included)  */
    int64_t interactions_pc; /* I_pc = sum_b count[b] * len_pc[b]                                */
    int64_t tiles_pp;        /* sum_b ceil(len_pp[b] / 32)                                       */
    int64_t tiles_pc;
    int64_t bad_entries;     /* validation failures (0 when the input is well-formed)            */
    int64_t chunks;          /* streamed variants: number of chunks issued, else 1              */
    int64_t fixup_sinks;     /* sinks re-evaluated by the fp64 fix-up kernel                      */
    int64_t invalid_values;  /* PKDG_VALIDATE: particles / cell records with values out of range  */
    int64_t invalid_pairs;   /* PKDG_VALIDATE: listed (sink, cell) pairs with |x - COM| <= b_max   */
    int64_t interactions_cc; /* pkdg_gravity_eval_fmm: entries of the C-C lists (one per bucket x cell)  */
    int64_t interactions_cp; /* pkdg_gravity_eval_fmm: entries of the C-P lists (one per bucket x particle) */
} pkdg_stats;

/* Create / destroy a context on CUDA device `device`.  The context owns only internal workspace
 * (normalised cell records, bucket descriptors, counters, staging buffers); it grows on demand
 * (the first call with a larger problem allocates and is therefore synchronous). */
pkdg_status pkdg_create(pkdg_ctx **ctx, int device);
pkdg_status pkdg_destroy(pkdg_ctx *ctx);

/* Options of a context.  PKDG_OPT_KAPPA2: conditioning threshold of the fp64 fix-up (> 0; default 6). */
#define PKDG_OPT_KAPPA2 1
pkdg_status pkdg_set_option(pkdg_ctx *ctx, int32_t option, double value);

/* One pass of the whole hot path with everything resident on the device:
 *   a1 packer       bucket work descriptors, tile counts, validation, I_pp / I_pc
 *   (cell prep)     canonical raw-moment records -> internal normalised trace-free records
 *   a2 staging, a3 P-P, a4 P-C, a5 reduction + write-back: one fused kernel, one warp per bucket
 * out_acc_pot = [particles->n][4] fp32 (ax, ay, az, phi), 16-byte aligned.  Rows of particles in a
 * listed bucket are overwritten (added to with PKDG_ACCUMULATE); other rows are untouched.
 * No host synchronisation once the workspace is large enough. */
pkdg_status pkdg_gravity_eval(pkdg_ctx *ctx, const pkdg_particles *particles, const pkdg_cells *cells,
                              const pkdg_buckets *buckets, const pkdg_list *pp, const pkdg_list *pc,
                              float eps, uint32_t flags, float *out_acc_pot, void *stream);

/* The same for the contiguous bucket range [b0, b1) of `buckets` (multi-GPU: every rank evaluates its own
 * range; no collective on the data path).  pp / pc hold the lists of those b1 - b0 buckets
 * only: b1 - b0 + 1 offsets, offsets[k] indexing `idx` as passed.  With PKDG_PP_LEAVES the references still
 * index the FULL `buckets` arrays.  pkdg_stats counts the range only. */
pkdg_status pkdg_gravity_eval_range(pkdg_ctx *ctx, const pkdg_particles *particles, const pkdg_cells *cells,
                                    const pkdg_buckets *buckets, int64_t b0, int64_t b1, const pkdg_list *pp,
                                    const pkdg_list *pc, float eps, uint32_t flags, float *out_acc_pot,
                                    void *stream);

/* The same with group-shared lists: pp / pc hold one list per GROUP (groups->n + 1 offsets).  A group's own
 * particles are on its P-P list like any others (self pairs are skipped by index).  4 x fewer list entries
 * to store and move than per-bucket lists; pkdg_stats counts sink x entry interactions as always. */
pkdg_status pkdg_gravity_eval_groups(pkdg_ctx *ctx, const pkdg_particles *particles, const pkdg_cells *cells,
                                     const pkdg_buckets *buckets, const pkdg_groups *groups, const pkdg_list *pp,
                                     const pkdg_list *pc, float eps, uint32_t flags, float *out_acc_pot,
                                     void *stream);

/* pkdg_gravity_eval for callers that must not allocate device memory.
 *
 * Who that is.  A pkdg_ctx buys its workspace with cudaMalloc (pkdg_create, and again whenever a call brings a
 * larger problem: "grows on demand" above, which also means a cudaFree).  Some hosts cannot live with that:
 *   - a simulation that hands out ALL device memory itself at start-up and leaves nothing for a library to take
 *     later (PKDGRAV3 pre-partitions its memory in just this way) -- a cudaMalloc in the middle of a
 *     run fails there, or succeeds and starves the owner;
 *   - a time-step loop that keeps several streams busy: cudaMalloc and cudaFree synchronise the whole device, so one
 *     workspace growth stalls every stream, not just ours;
 *   - code that runs where the CUDA allocator may not be called at all (a stretch of the program its authors have
 *     declared allocation-free, for predictability or because it sits inside another library's callback).
 * This entry point needs no pkdg_ctx and calls neither cudaMalloc nor cudaFree nor any CUDA routine that allocates:
 * the bucket descriptors, the normalised cell records, the fp64 fix-up queue and the counters that the kernels of
 * pkdg_gravity_eval keep in the context's workspace live here in one fixed array in device memory that is part of
 * the library image (a file-scope `static __device__` array in pkdg.cu, PKDG_STATIC_SCRATCH_BYTES ~ 6.1 MB).  The
 * price: every GPU on which this library's code is loaded holds those bytes until the process exits, whether or
 * not this function is ever called, and the problem size is capped:
 *     buckets->n <= PKDG_STATIC_MAX_BUCKETS, cells->n <= PKDG_STATIC_MAX_CELLS,
 *     particles->n <= PKDG_STATIC_MAX_PARTICLES;
 * anything larger is refused with PKDG_EINVAL and a text that names the limit (nothing is queued).  Cut a larger
 * problem into bucket ranges yourself, or use a pkdg_ctx.
 *
 * Arguments, layouts, results and stream behaviour are those of pkdg_gravity_eval (the same kernels run; rows
 * are bit-identical to it): all pointers are device pointers on `device`, the caller owns inputs and `out_acc_pot`,
 * the call is asynchronous on `stream`.  Flags: PKDG_ACCUMULATE, PKDG_SKIP_PP, PKDG_SKIP_PC, PKDG_NO_FIXUP,
 * PKDG_FIXUP_ALL; PKDG_PP_LEAVES and PKDG_VALIDATE need workspace of their own and are refused.  The fix-up
 * threshold is the default kappa2 = 6.  There are no counters to read back (pkdg_get_stats needs a context):
 * malformed buckets or list entries are skipped as in pkdg_gravity_eval but not reported -- validate the inputs
 * once through a context if they come from an untrusted builder.
 *
 * First call on a device.  The first call for a given `device` (from any thread) looks up the device address of
 * the array (on the host the array's name is only a handle, not an address a kernel could use), the SM count and
 * the kernel's shared-memory opt-in, with that device current, and remembers them.  It allocates nothing either,
 * but it does talk to the driver: make that first call once, early, outside any stream capture.  Later calls only
 * queue two memsets and four kernels.
 *
 * Sharing.  There is ONE array per device and every call on that device uses it, from every thread and every
 * stream.  It still holds what the previous call left; each call clears the counters it needs at zero itself
 * (stream-ordered, before its kernels) and overwrites every descriptor, record and queue entry before reading it,
 * so back-to-back calls on one stream are safe.  Two calls whose GPU work may OVERLAP (different streams without
 * an event between them, or two host threads) race on the array and give wrong rows: order them.  Calls made
 * through a pkdg_ctx need no such care: a context has its own workspace and never touches the array.
 * Errors: PKDG_EINVAL (arguments, limits, flags), PKDG_ECUDA; the text is at pkdg_last_error(NULL). */
#define PKDG_STATIC_MAX_BUCKETS 32768
#define PKDG_STATIC_MAX_CELLS 32768
#define PKDG_STATIC_MAX_PARTICLES 524288
#define PKDG_STATIC_SCRATCH_BYTES (512 + 32 * PKDG_STATIC_MAX_BUCKETS + 128 * PKDG_STATIC_MAX_CELLS + \
                                   16 * (PKDG_STATIC_MAX_BUCKETS + PKDG_STATIC_MAX_PARTICLES / 16 + 16))
pkdg_status pkdg_gravity_eval_static(int device, const pkdg_particles *particles, const pkdg_cells *cells,
                                     const pkdg_buckets *buckets, const pkdg_list *pp, const pkdg_list *pc,
                                     float eps, uint32_t flags, float *out_acc_pot, void *stream);

/* The FMM form of the path (PAPER.md:L57 cell-cell interactions, L69 fn 2 cell-particle
 * interactions, L71 "The local expansion of the potential about the sink's center of mass is actually done to
 * 5th order ... accumulating the CC and CP interactions"; readings A20-A22).  Every bucket b has four
 * lists: pp and pc as in pkdg_gravity_eval, plus cc (indices of source CELLS) and cp (indices of source
 * PARTICLES) that act on the bucket as a whole through its local expansion about centres[b] ([n_buckets][3]
 * fp32, device; the bucket's centre of mass in the paper):
 *     L_n = - sum_m (-1)^|m| M_m binom(n+m, m) t_{n+m}(centres[b] - COM_c),  |n| <= 5,  |n| + |m| <= 5,
 *           |m| in {0, 2, 3, 4}  (a source particle is a cell with only M_0 = m_j at x_j),
 *     phi_i += sum_n L_n s^n,   a_i -= grad of that polynomial,   s = x_i - centres[b],
 * t_k = d^k(1/|r|)/k! as above; unsoftened.  The result is the SUM of the four lists' contributions.  Any of the
 * four lists may be NULL.  A C-C or C-P source must lie outside the sphere of the bucket's sinks about
 * centres[b] (the expansion diverges inside; any acceptance criterion of the kind of PAPER.md:L69 ensures it).
 * PKDG_PP_LEAVES is not supported here.  pkdg_stats: interactions_cc / interactions_cp count list entries. */
pkdg_status pkdg_gravity_eval_fmm(pkdg_ctx *ctx, const pkdg_particles *particles, const pkdg_cells *cells,
                                  const pkdg_buckets *buckets, const float *centres, const pkdg_list *pp,
                                  const pkdg_list *pc, const pkdg_list *cp, const pkdg_list *cc, float eps,
                                  uint32_t flags, float *out_acc_pot, void *stream);

/* Streamed variant (a6; "fully asynchronous", L278 bounded queue): particles, cells
 * and out are device buffers, buckets and lists are PINNED HOST buffers.  Contiguous bucket ranges
 * ("chunks", greedy fill to at most max_entries_per_chunk P-P and P-C entries; a longer single
 * bucket forms its own chunk) are copied host->device and evaluated round-robin on n_streams
 * internal streams; at most n_streams chunks are in flight.  Returns after the last chunk has been
 * queued; `stream` waits for all of them. */
pkdg_status pkdg_gravity_eval_streamed(pkdg_ctx *ctx, const pkdg_particles *particles,
                                       const pkdg_cells *cells, const pkdg_buckets *buckets_host,
                                       const pkdg_list *pp_host, const pkdg_list *pc_host, float eps,
                                       uint32_t flags, float *out_acc_pot, int32_t n_streams,
                                       int64_t max_entries_per_chunk, void *stream);

/* End-to-end variant: EVERY buffer is a host buffer (pinned for full speed).  Copies particles and
 * cells to the device, streams the lists as above, copies the result back into out_acc_pot_host and
 * synchronises before returning (also when it returns an error).  Rows of particles in no listed bucket
 * keep the caller's values, as in pkdg_gravity_eval.  When every bucket starts where the previous one
 * ends (the tree order of PAPER.md:L63) the rows of each chunk are copied back on the chunk's stream as
 * soon as its kernels are done, overlapping the host->device traffic of later chunks; otherwise the
 * caller's rows make a round trip through the device.
 * pkdg_gravity_eval_host_range: the same for the bucket range [b0, b1) of `buckets_host`, with the lists
 * of that range only (multi-GPU end to end: each rank passes its own range and lists).
 * pkdg_gravity_eval_host_groups: the same with group-shared lists (chunks are then ranges of groups). */
pkdg_status pkdg_gravity_eval_host(pkdg_ctx *ctx, const pkdg_particles *particles_host,
                                   const pkdg_cells *cells_host, const pkdg_buckets *buckets_host,
                                   const pkdg_list *pp_host, const pkdg_list *pc_host, float eps,
                                   uint32_t flags, float *out_acc_pot_host, int32_t n_streams,
                                   int64_t max_entries_per_chunk);
pkdg_status pkdg_gravity_eval_host_groups(pkdg_ctx *ctx, const pkdg_particles *particles_host,
                                          const pkdg_cells *cells_host, const pkdg_buckets *buckets_host,
                                          const pkdg_groups *groups_host, const pkdg_list *pp_host,
                                          const pkdg_list *pc_host, float eps, uint32_t flags,
                                          float *out_acc_pot_host, int32_t n_streams,
                                          int64_t max_entries_per_chunk);
pkdg_status pkdg_gravity_eval_host_range(pkdg_ctx *ctx, const pkdg_particles *particles_host,
                                         const pkdg_cells *cells_host, const pkdg_buckets *buckets_host,
                                         int64_t b0, int64_t b1, const pkdg_list *pp_host,
                                         const pkdg_list *pc_host, float eps, uint32_t flags,
                                         float *out_acc_pot_host, int32_t n_streams,
                                         int64_t max_entries_per_chunk);

/* List construction on the device.  The tree as the walk needs it, all arrays on
 * the device, cells in depth-first pre-order ("hierarchically sorted"): cell k's subtree is
 * cells [k, end[k]), its first child is k + 1; first / count = its particle run; isleaf != 0 marks a bucket;
 * bblo / bbhi = [n_cells][3] bounding boxes of the fp32 coordinates; the centre of mass and
 * b_max come from the canonical cell records.  leaf_rank (may be NULL) = [n_cells], bucket index of a leaf. */
typedef struct {
    const int32_t *first, *count, *end, *isleaf;
    const float *bblo, *bbhi;
    const int32_t *leaf_rank;
    int64_t n_cells;
} pkdg_tree;

/* The tree walk that resolves a sink cell's checklist into its P-P and P-C list (the
 * acceptance test is DESIGN.md reading A6: cell k is a P-C source for sink B iff k != B, it holds >= 2
 * particles, |COM_B - COM_k| > b_max,B + b_max,k / theta and the bounding boxes are >= 2 eps apart; a leaf
 * that fails joins the P-P list whole; any other cell is opened).  sink_cell[n_sinks] names the sink cells:
 * the leaf cells for per-bucket lists, the group cells for group-shared lists.  Two calls, because the caller
 * owns the index arrays: _count writes the CSR offsets (n_sinks + 1 each, device) and returns the two totals
 * in totals_host[2] (synchronises; NULL = stay asynchronous); _fill writes the entries, in walk order.  With
 * PKDG_PP_LEAVES a P-P entry is the bucket index of the leaf instead of its particles.  Decisions are taken in
 * fp64 with IEEE operations and no contraction: offsets and indices are bit-identical to a host walk.
 * Malformed tree input does not hang or read out of bounds: an end[k] outside (k, n_cells] is clamped into it and
 * a sink_cell outside [0, n_cells) gets two empty lists; both are counted in pkdg_stats.bad_entries, which
 * pkdg_get_stats reports (PKDG_EBADLIST) when called after _count and before the next evaluation call. */
pkdg_status pkdg_build_lists_count(pkdg_ctx *ctx, const pkdg_tree *tree, const pkdg_cells *cells,
                                   const int32_t *sink_cell, int64_t n_sinks, double theta, double eps,
                                   uint32_t flags, int64_t *pp_offsets, int64_t *pc_offsets,
                                   int64_t *totals_host, void *stream);
pkdg_status pkdg_build_lists_fill(pkdg_ctx *ctx, const pkdg_tree *tree, const pkdg_cells *cells,
                                  const int32_t *sink_cell, int64_t n_sinks, double theta, double eps,
                                  uint32_t flags, const int64_t *pp_offsets, const int64_t *pc_offsets,
                                  int32_t *pp_idx, int32_t *pc_idx, void *stream);

/* End to end from the TREE (every buffer on the host, pinned for full speed): the lists are built on the device
 * (pkdg_build_lists_*, P-P entries as bucket references) and evaluated, so only particles, cells and the tree cross the
 * bus, not the lists.  tree_host holds host arrays (leaf_rank is ignored); buckets_host are ALL the leaves of the tree
 * as sinks, contiguous runs of particles in ascending order, and bucket_cell_host[b] is the leaf cell of
 * bucket b (a P-P source leaf is named by its bucket index, so a subset of the leaves is refused with PKDG_EINVAL; for
 * a subset of sinks use pkdg_build_lists_* and pkdg_gravity_eval_range).
 * Tree, cells and buckets are copied first; the walk runs while the particles are still arriving; the evaluation is
 * cut into n_ranges (1..64; 4 is a good value) bucket ranges and the rows of a range are copied back while the next
 * range is evaluated.  Synchronous; rows of particles in no bucket keep the caller's values.  Flags: PKDG_NO_FIXUP,
 * PKDG_FIXUP_ALL, PKDG_VALIDATE.  pkdg_stats holds the totals of the call (chunks = n_ranges). */
pkdg_status pkdg_gravity_eval_tree_host(pkdg_ctx *ctx, const pkdg_particles *particles_host, const pkdg_cells *cells_host,
                                        const pkdg_tree *tree_host, const pkdg_buckets *buckets_host,
                                        const int32_t *bucket_cell_host, double theta, float eps, uint32_t flags,
                                        float *out_acc_pot_host, int32_t n_ranges);

/* Packer made visible for bit-exact checks (SURVEY.md sec 8(c) "Integer side"): the tiles the
 * evaluation kernel consumes.  tile_offsets = [n_buckets+1] int64 (first tile of each bucket);
 * tiles = [tile_capacity][32] int32, list order, last tile of a bucket padded with PKDG_PAD.
 * Either output may be NULL.  If the list needs more than tile_capacity tiles only tile_offsets is
 * complete (tile_offsets[n_buckets] is the number needed). */
pkdg_status pkdg_pack_export(pkdg_ctx *ctx, int64_t n_buckets, const pkdg_list *list,
                             int64_t *tile_offsets, int32_t *tiles, int64_t tile_capacity, void *stream);

/* Chunk boundaries the streamed variants use, from HOST offsets: bounds_host gets n_chunks+1
 * values (room for n_buckets+1); *n_chunks_host the count.  Pure host code. */
pkdg_status pkdg_chunk_bounds(int64_t n_buckets, const int64_t *pp_offsets_host,
                              const int64_t *pc_offsets_host, int64_t max_entries_per_chunk,
                              int64_t *bounds_host, int64_t *n_chunks_host);

/* Internal normalised cell records made visible for tests: out = [cells->n][32] fp32. */
pkdg_status pkdg_prepare_cells_export(pkdg_ctx *ctx, const pkdg_cells *cells, float *out, void *stream);

/* Synchronises the stream(s) of the last evaluation and returns its counters. */
pkdg_status pkdg_get_stats(pkdg_ctx *ctx, pkdg_stats *stats_host);

/* Device timing of the evaluation kernel alone (the dominant kernel of the path) and of the fp64 fix-up
 * kernel that follows it.  With profiling on, pkdg_gravity_eval(_range) brackets those launches with CUDA
 * events on the launching stream (ring of 256 calls).  pkdg_profile_read synchronises, returns the number
 * of calls recorded since the last read and the total duration of each kernel in milliseconds
 * (fixup_ms_total_host may be NULL), and clears the ring. */
pkdg_status pkdg_profile_enable(pkdg_ctx *ctx, int32_t on);
pkdg_status pkdg_profile_read(pkdg_ctx *ctx, int64_t *n_launches_host, double *eval_ms_total_host,
                              double *fixup_ms_total_host);

/* Number of kernel launches this context has made since creation. */
int64_t pkdg_launch_count(const pkdg_ctx *ctx);

const char *pkdg_status_string(pkdg_status s);
/* Text of the last error on ctx; with ctx == NULL, why the calling thread's last pkdg_create or
 * pkdg_gravity_eval_static failed (the two calls that have no context to hold the text). */
const char *pkdg_last_error(const pkdg_ctx *ctx);
void pkdg_version(int32_t *major, int32_t *minor);

/* FP32 FFMA-only micro-benchmark (roofline denominator check): runs `iters` dependent-chain-free
 * FFMA rounds on every SM and returns the elapsed milliseconds and the flop count. Synchronous. */
pkdg_status pkdg_fma_peak_probe(pkdg_ctx *ctx, int64_t iters, float *ms_host, double *flops_host);

#ifdef __cplusplus
}
#endif
#endif /* PKDG_H */
