/*
 * comet.h -- C ABI of the B200-native seed x hit scan of arXiv 1911.09340
 * ("GPU-accelerated event reconstruction for the COMET Phase-I experiment").
 *
 * Citations are /root/reference/PAPER.md line numbers; R<n> are the readings listed in
 * DESIGN.md section 2.  Units: cm, MeV/c, Tesla, charge in units of e.
 *
 * Conventions
 *   - Every function returns COMET_OK (0) or a negative comet_status.  Nothing throws.
 *   - "dev" pointers are CUDA device memory owned by the caller, 16-byte aligned, valid until
 *     the work enqueued on `cuda_stream` has completed.  "host" pointers are ordinary host
 *     memory read or written before the call returns unless stated otherwise.
 *   - `cuda_stream` is a cudaStream_t cast to void* (NULL = the legacy default stream).
 *     The device-buffer calls only enqueue work: no host synchronisation, and no allocation once the
 *     ctx's workspace has been sized (comet_reserve_scan / comet_reserve; a call that finds it too small
 *     grows it -- that call synchronises the device -- unless the stream is being captured into a CUDA
 *     graph, where it returns COMET_ENOMEM instead).  The entry points that say so (the turn loops, the
 *     host-buffer calls, comet_seed_runs) synchronise the stream.
 *   - A comet_ctx owns a small device workspace; use one ctx per stream.  Calls on different
 *     ctx objects / streams are independent.
 *   - There is no CPU implementation behind this interface.
 */
#ifndef COMET_H_
#define COMET_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct comet_ctx comet_ctx;

typedef enum comet_status {
    COMET_OK = 0,
    COMET_EINVAL = -1,   /* null pointer, negative size, bad option, limits exceeded */
    COMET_ENOMEM = -2,   /* device or host allocation failed */
    COMET_ECUDA = -3,    /* a CUDA runtime call failed; see comet_last_cuda_error */
    COMET_ELIMIT = -4    /* comet_argmin_static: more partitions than its statically allocated scratch holds */
} comet_status;

/* Seeds per track chunk: the track buffer is laid out in chunks of 32 consecutive seeds
 * (one warp of lanes), see comet_track_bytes. */
#define COMET_CHUNK 32
/* Limits checked by the entry points. */
#define COMET_MAX_PARTITIONS 64
#define COMET_MAX_STEPS 4096

/* Options for comet_set_option. */
#define COMET_OPT_COARSE_SEARCH 1     /* how step B2 (closest recorded state) is found          */
#define COMET_COARSE_EXHAUSTIVE 0     /*   every recorded state is evaluated for every wire         */
#define COMET_COARSE_PRUNED 1         /*   default: block samples + Lipschitz bounds skip states that cannot be
                                       *   the closest one, and (when neither dca nor kstar is requested) pairs
                                       *   whose residual is provably the cutoff; k*, D and rss are identical   */
#define COMET_OPT_TIMING 3            /* 1: comet_dca_rss (pruned) times its kernels, see comet_read_timing      */
#define COMET_OPT_LANES 4             /* 1..8 (default 6, 4 with COMET_OPT_ZGROUP): sub-slabs comet_scan_rss runs concurrently on internal streams */
#define COMET_OPT_ZGROUP 5            /* 1 (default): comet_scan_rss steps every distinct transverse track once when runs of >= 8
                                       *   consecutive seeds differ only in z (found on the device; results are identical) and the
                                       *   call has at least 1024 chunks; 2: whatever the size of the call; 0: never */
#define COMET_OPT_STATS 2             /* 1: comet_dca_rss (pruned) adds its work counters, see comet_read_stats  */

/* ---- context ---------------------------------------------------------------------------- */

/* Creates a context on CUDA device `cuda_device` (allocates a few MB of device workspace). */
int comet_create(comet_ctx** out, int cuda_device);
/* Frees the workspace.  The caller must have synchronised every stream that used the ctx. */
int comet_destroy(comet_ctx* ctx);
/* Static, never freed. */
const char* comet_status_string(int status);
/* cudaError_t of the last failing CUDA call made through this ctx (0 if none). */
int comet_last_cuda_error(const comet_ctx* ctx);
int comet_set_option(comet_ctx* ctx, int option, int value);
int comet_get_option(const comet_ctx* ctx, int option, int* value);

/* Sets the size of the (seed, wire) pair workspace of the pruned search to max_pairs_per_launch
 * pairs (8 bytes each, 12 on the materialised path; default limit 2^29) and allocates it now, so that later comet_dca_rss calls
 * never allocate.  comet_dca_rss processes larger problems in seed slabs that fit; without this
 * call the workspace grows on the first comet_dca_rss that needs it (that call synchronises the
 * device). */
int comet_reserve(comet_ctx* ctx, int64_t max_pairs_per_launch);

/* Sizes every workspace comet_scan_rss (and the calls built on it: comet_scan_stage, comet_scan_turns, the
 * half-track calls) needs for seed sets of up to n_seeds seeds (with the z_run the scans will promise, and for
 * calls without a promise), n_steps steps and n_fired fired wires --
 * (seed, wire) pair keys, checkpoints, per-seed constants, the distinct-track rows of the z-run kernels --
 * under the current options and field mode, so that those calls never allocate or synchronise afterwards
 * (they can then be captured into a CUDA graph from the first call on).  Larger problems than comet_reserve's
 * pair limit (default 2^29 pairs) or 8 GiB of checkpoints allow are processed in seed slabs of that size: with
 * the run length promised a checkpoint is one z per seed and 8 states, without it (x, T) per seed and 4 states,
 * so a promised configs[3] scan is one slab and an unpromised one ten.  Synchronises the device when it
 * reallocates. */
int comet_reserve_scan(comet_ctx* ctx, int64_t n_seeds, int32_t z_run, int32_t n_steps, int32_t n_fired);

/* With COMET_OPT_TIMING = 1 the pruned comet_dca_rss and comet_scan_rss record CUDA events on the caller's
 * stream around their kernels (once per seed slab; comet_scan_rss then runs its sub-slabs one after the other).
 * Waits for the timed slabs and writes the mean device time in milliseconds over the most recent ones (at most
 * 64 since the option was set or the last read) to ms_host[0..n), n <= 4 -- [0] the closest-state search
 * (k_coarse_pruned / k_scan_fused / k_scan_zrun), [1] the fine stage (k_fine / k_fine_ck), [2] k_rss_sum,
 * [3] k_gen_unique (0 when the z-run kernels did not serve the call) --, their number to *n_calls (may be NULL),
 * and restarts the count.  COMET_EINVAL if no timed call was made. */
int comet_read_timing(comet_ctx* ctx, float* ms_host, int32_t n, int32_t* n_calls);

/* Copies the work counters accumulated by comet_dca_rss calls made with COMET_OPT_STATS = 1 to
 * out_host[0..n) (HOST, n <= 9) and synchronises the stream; reset != 0 zeroes them afterwards.
 * Counters are thread-level: [0] block/sub-block sample evaluations, [1] row evaluations a lane
 * needed, [2] row evaluations executed (a warp opens a sub-block when any lane needs it),
 * [3] (seed, wire) pairs that needed the virtual-plane iteration, [4] pairs for which a warp
 * executed it, [5] all pairs, [6] RKN4 steps of distinct transverse tracks (comet_scan_rss with
 * COMET_OPT_ZGROUP; 0 otherwise), [7] tangent-line tests of k_scan_zrun's level B (per wire, sub-block and
 * distinct track; [0] then counts its level-A samples), [8] 32 x (chunk, wire) key rows it created. */
int comet_read_stats(comet_ctx* ctx, uint64_t* out_host, int32_t n, int32_t reset, void* cuda_stream);

/* ---- inhomogeneous field map and adaptive step (R29-R32) ------- */

#define COMET_MAX_STEPS_FIELD 4000    /* n_steps limit while a field map is set */

/* "BFields in the grid format": field_dev is a regular grid [nx][ny][nz][3] of
 * (Bx, By, Bz) in Tesla (dev, caller-owned, must stay valid while it is set), node (i,j,k) at
 * origin_cm + (i dx, j dy, k dz); n_nodes, origin_cm, spacing_cm are HOST [3].  The field at a point
 * is the trilinear interpolation, the edge value outside the grid (R29).  While a map is set,
 * comet_scan_rss, comet_select_and_classify, comet_classify_seeds, comet_scan_stage and
 * comet_scan_event_host (fused) extrapolate in it -- their bz_tesla argument is ignored -- with the
 * Nystrom RK4 step of R30 and the adaptive step of R31 ("an adaptive step size that adjusts to the
 * roughness of the magnetic field"): step_cm is the longest step h_max, a step whose
 * error estimate exceeds rkn_tol_cm is retried with half the length (not below h_max/64), after a
 * step with an estimate below rkn_tol_cm/32 the next trial step doubles; n_steps stays the capacity
 * in recorded states (<= COMET_MAX_STEPS_FIELD).  comet_seed_extrapolate and comet_dca_rss (the
 * materialised track) are uniform-field paths and return COMET_EINVAL.  field_dev = NULL returns
 * to the uniform field.  Enqueues one small kernel on cuda_stream (the map's largest |B|). */
int comet_set_field(comet_ctx* ctx, const double* field_dev, const int32_t* n_nodes,
                    const double* origin_cm, const double* spacing_cm, double rkn_tol_cm,
                    void* cuda_stream);

/* ---- kernel A: track recording (Algorithm 1) ---------------------------- */

/* Bytes of the opaque track buffer for n_seeds seeds and n_steps steps.
 * Layout (library-defined): two planes, positions X then unit tangents T, each
 * [n_chunks][R][3][32] doubles with n_chunks = ceil(n_seeds/32) and R = n_steps+1 rounded up to
 * a multiple of 64: component c of recorded state k of seed s is at ((s/32 * R + k) * 3 + c) * 32
 * + s%32.  Position rows between a seed's last state and the end of its chunk's last 64-row block
 * repeat the last state (padding read by kernel B).
 * Returns 0 for invalid arguments. */
size_t comet_track_bytes(int64_t n_seeds, int32_t n_steps);

/* Every seed (x,p)_0 is extrapolated as a charged particle in the uniform field (0,0,bz):
 * T_0 = p/|p|, c = kappa*charge*bz/|p| (kappa = 2.99792458, R4), then n_steps classical
 * Runge-Kutta-Nystrom steps of length step_cm (R1, R2), every state recorded
 * (PAPER.md:138).  Recording stops at the first recorded state inside the target region
 * r < r_stop_cm and moving inward (R3); r_stop_cm = 0 never stops.
 *   seeds       dev, SoA: component j (x,y,z,px,py,pz) of seed s at seeds[j*seed_stride + s]
 *   seed_stride distance in doubles between components (>= n_seeds)
 *   track       dev, comet_track_bytes(n_seeds, n_steps) bytes, written
 *   n_pts       dev [n_seeds], written: number of recorded states, 2..n_steps+1
 * Arithmetic: fp64, one IEEE operation per operation of the definition (no contraction). */
int comet_seed_extrapolate(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                           int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                           double r_stop_cm, void* track, int32_t* n_pts, void* cuda_stream);

/* Copies seeds [seed_begin, seed_end) of a track buffer to the canonical layout
 * out[(s - seed_begin)][k][6] = x,y,z,Tx,Ty,Tz (dev), NaN for k >= n_pts[s]. */
int comet_track_export(comet_ctx* ctx, const void* track, const int32_t* n_pts, int64_t n_seeds,
                       int32_t n_steps, int64_t seed_begin, int64_t seed_end, double* out,
                       void* cuda_stream);

/* ---- kernel B: DCA finding and RSS (Algorithm 2; Eq. (1), :75-77) -------- */

/* For every seed s and fired wire i: the recorded state closest to the wire line (R5, R6;
 * PAPER.md:165), the virtual-plane iteration with RKN sub-steps from it (R7-R10; PAPER.md:167-184,
 * :216), the signed distance of closest approach D (R16); then
 *   rss[s] = sum_i min( min_{j in [hit_off[i], hit_off[i+1])} |D - rho[j]|, cutoff )^2
 * accumulated in increasing i (Eq. (1); a wire without entries contributes cutoff^2).
 *   track, n_pts   as written by comet_seed_extrapolate with the same n_seeds, n_steps,
 *                  charge, bz_tesla, step_cm
 *   wire_a, wire_b dev, SoA [3][n_wires]: wire endpoints
 *   fired_wire     dev [n_fired]: indices into the wire table of the wires that have hits (R11)
 *   hit_off        dev [n_fired+1]: CSR offsets into rho, non-decreasing, hit_off[n_fired] = n_hits
 *   rho            dev [n_hits]: signed drift distance of each hit entry, +r and -r for the
 *                  left/right ghosts (R12)
 *   rss            dev [n_seeds], written
 *   dca            dev [n_seeds][n_fired] signed D, written; NULL to skip
 *   kstar          dev [n_seeds][n_fired] index of the closest recorded state; NULL to skip */
int comet_dca_rss(comet_ctx* ctx, const void* track, const int32_t* n_pts, int64_t n_seeds,
                  int32_t n_steps, int32_t charge, double bz_tesla, double step_cm,
                  const double* seeds, int64_t seed_stride,
                  const double* wire_a, const double* wire_b, int32_t n_wires,
                  const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                  int32_t n_fired, int32_t n_hits, double cutoff_cm,
                  double* rss, double* dca, int32_t* kstar, void* cuda_stream);

/* ---- kernels A + B fused, track kept on chip (Algorithms 1 + 2) ------------ */

/* rss[s] (and n_pts[s]) exactly as comet_seed_extrapolate followed by comet_dca_rss(dca = kstar =
 * NULL) would produce them -- same operations, bit-identical -- but the recorded track never goes
 * to HBM: a warp extrapolates a chunk of 32 seeds tile by tile into shared memory, searches the
 * tile for the states closest to every fired wire, and keeps only every 4th recorded state in a
 * checkpoint workspace from which the virtual-plane iteration restarts.
 * Arguments as in the two calls above;
 *   n_pts   dev [n_seeds], written; NULL to skip.
 * Workspace (checkpoints: 12 bytes per recorded state of capacity; 8 bytes per (seed, wire) pair;
 * 8 bytes per seed) lives in the ctx: sized by comet_reserve_scan, else grown on the first call that
 * needs it (that call synchronises the device; COMET_ENOMEM while the stream is being captured); larger problems are processed in seed slabs bounded by comet_reserve's
 * pair limit and by 8 GiB of checkpoints.  A slab is cut into up to COMET_OPT_LANES sub-slabs that
 * run concurrently on streams owned by the ctx; `cuda_stream` forks into them and joins them again
 * with events, so the call is asynchronous with respect to the host and ordered on `cuda_stream`
 * like any other work (and can be captured into a CUDA graph).  COMET_OPT_TIMING (k_scan_fused,
 * k_fine_ck, k_rss_sum) and COMET_OPT_STATS run the sub-slabs one after the other on `cuda_stream`.
 * With COMET_OPT_STATS the counters of comet_read_stats mean: [0] sub-block samples evaluated
 * (one per wire, sub-block and chunk), [1] rows swept for a lane whose tile holds recorded states,
 * [2] rows swept, [3] pairs that needed the virtual-plane iteration, [4] 32 x (chunk, wire) items
 * for which a warp executed it, [5] all pairs, [6] RKN4 steps taken for distinct transverse tracks
 * by the z-run kernels (0 when the plain kernels served the call).
 * COMET_OPT_ZGROUP (default 1, uniform field only): in B = (0, 0, B_z) the transverse motion does
 * not depend on z, so seeds with bit-identical (x, y, p_x, p_y, p_z) share their (x, y, T_x, T_y)
 * sequence and their stop.  When every aligned run of ZG >= 8 consecutive seeds of the call is
 * uniform in those components (found on the device; the seed grids of the method with z as the
 * fastest axis are), the RKN4 steps are taken once per distinct transverse track and every seed
 * adds its own z column; rss and n_pts are the same numbers either way.  Calls of fewer than 1024
 * chunks (32768 seeds) always take the plain kernels.
 *   z_run   what the caller knows about the seeds: 0 = nothing (the run length is found on the device: one
 *           small kernel per sub-slab, and both kernel variants are enqueued, the one that does not serve
 *           the launch returns at once); 8, 16, 32, ... (a power of two) = a promise that every aligned run
 *           of min(z_run, 32) consecutive seeds, counted from seeds[0], is bit-identical in (x, y, p_x, p_y,
 *           p_z) -- comet_seed_grid's output with z_run = comet_grid_z_run(n_z), or what comet_seed_runs
 *           found; a false promise gives wrong results, it is not checked; 1 = no runs: plain kernels.
 * Workspace: see comet_reserve_scan. */
int comet_scan_rss(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                   int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                   const double* wire_a, const double* wire_b, int32_t n_wires,
                   const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                   int32_t n_fired, int32_t n_hits, double cutoff_cm,
                   double* rss, int32_t* n_pts, void* cuda_stream);

/* ---- step C: best seed per turn partition and hit classification -------- */

/* For every partition p (seeds [part_off[p], part_off[p+1])): best_seed[p] = lowest-index argmin
 * of rss (R15), best_rss[p] its value.  That seed is extrapolated again and, on every fired wire,
 * the hit entry closest to its D (ties -> lowest index) is classified iff |D - rho| < cutoff
 * (R13): cls[p][j] = 1, all other entries 0.  best_dca[p][i] = D.
 *   part_off   HOST [n_part+1], non-decreasing, within [0, n_seeds]; read before returning
 *   best_seed  dev [n_part] (global seed index, -1 for an empty partition), best_rss dev [n_part],
 *   best_dca   dev [n_part][n_fired], cls dev [n_part][n_hits]
 * A NaN in rss follows the serial rule "rss[s] < rss[best]": it wins only at the first seed of a partition.
 * When the last comet_scan_rss of this ctx scanned exactly this seed set (same buffer, stride, count and physics,
 * uniform field, one slab), the winner's track is not stepped again as one chain of n_steps dependent steps: with
 * z_run promised its (x, y, T_x, T_y) rows are copied from that scan's distinct-track workspace; after the plain
 * kernels (small sets, z_run = 1) every 4th recorded state is that scan's checkpoint and the three states after
 * it are stepped by one thread per checkpoint -- the same numbers either way.  A reused track is checked on the
 * device: its state 0 must equal the seed's own initial state bit for bit, else the track is stepped again (a
 * seed buffer rewritten in place, or handed out again by an allocator, is harmless).  The wire lines (O4) are
 * formed from wire_a / wire_b by the classifying kernel itself: nothing of an earlier call's hit list is used.
 * Partitions of at most 16384 seeds are searched by the classifying CTA itself (one launch).
 * Limits: n_part <= COMET_MAX_PARTITIONS, n_steps <= COMET_MAX_STEPS. */
int comet_select_and_classify(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                              int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                              double r_stop_cm,
                              const double* wire_a, const double* wire_b, int32_t n_wires,
                              const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                              int32_t n_fired, int32_t n_hits, double cutoff_cm,
                              const double* rss, const int64_t* part_off, int32_t n_part,
                              int64_t* best_seed, double* best_rss, double* best_dca, uint8_t* cls,
                              void* cuda_stream);

/* ---- iterative seed refinement (readings R24-R28 of DESIGN.md) ------ */

#define COMET_MAX_REFS 64             /* limit of k_ref and k_final */

/* "several seeds with the lowest RSS are selected as reference points for the next seed scanning
 * [...] sparse enough to avoid overlaps between new seed sets from each reference point"
 * (PAPER.md:81).  The refined components are (z, p_x, p_y, p_z) = seed components 2..5 at the
 * reference's (x, y) (R24).  Per partition p, ref_seed[p][0..k_ref) are taken one by
 * one: the seed of lowest rss (ties -> lowest index, NaN never) that is not selected yet and whose
 * box ref_d +- half_width[d] overlaps no selected box; two boxes overlap iff
 * |ref_a,d - ref_b,d| < 2 half_width[d] in every dimension d (R25).  -1 where no seed is left.
 *   rss         dev [n_seeds];  part_off  HOST [n_part+1];  half_width  HOST [4], >= 0
 *   ref_seed    dev [n_part][k_ref], written (global seed indices) */
int comet_select_references(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                            const double* rss, const int64_t* part_off, int32_t n_part,
                            const double* half_width, int32_t k_ref, int64_t* ref_seed,
                            void* cuda_stream);

/* "new seeds are fetched in their vicinity and with a finer granularity": slot
 * (p, r) of new_seeds holds G = n_grid[0] n_grid[1] n_grid[2] n_grid[3] seeds around reference
 * ref_seed[p][r] (an empty slot repeats ref_seed[p][0], R27): component 2+d takes the values
 * (ref_d - half_width[d]) + j (2 half_width[d] / (n_grid[d] - 1)), j = 0..n_grid[d]-1 (the
 * reference's own value when n_grid[d] = 1), (x, y) are the reference's; the seed of (j0..j3) is at
 * index ((j0 n1 + j1) n2 + j2) n3 + j3 of the slot, slot (p, r) starts at (p k_ref + r) G (R26).
 *   new_seeds   dev SoA [6][new_stride], new_stride >= n_part k_ref G, written
 *   n_grid      HOST [4], each 1..4096 */
int comet_refine_seeds(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                       const int64_t* ref_seed, int32_t n_part, int32_t k_ref,
                       const double* half_width, const int32_t* n_grid,
                       double* new_seeds, int64_t new_stride, void* cuda_stream);

/* The classification rule of PAPER.md:83 (as in comet_select_and_classify) for the listed seeds:
 * dca[n][i] = signed D of seed seed_idx[n] on fired wire i, cls[n][j] = 1 for the classified hit
 * entries.  seed_idx[n] < 0 gives NaN / zeros.
 *   seed_idx  dev [n_sel];  dca  dev [n_sel][n_fired];  cls  dev [n_sel][n_hits] */
int comet_classify_seeds(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                         int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                         double r_stop_cm,
                         const double* wire_a, const double* wire_b, int32_t n_wires,
                         const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                         int32_t n_fired, int32_t n_hits, double cutoff_cm,
                         const int64_t* seed_idx, int32_t n_sel, double* dca, uint8_t* cls,
                         void* cuda_stream);

/* Bytes of the device work buffer of comet_scan_stage (0 for invalid arguments). */
size_t comet_stage_work_bytes(int64_t n_seeds, int32_t n_part, int32_t k_ref, int32_t k_final,
                              const int32_t* n_grid);

/* One *stage* (the seed scanning of a turn, several *iterations*) for all turn
 * partitions at once, entirely on the device (the paper crosses the PCIe bus four times per
 * iteration).  Iteration 0: comet_scan_rss of the given seeds.  Each
 * of the n_iter further iterations: comet_select_references (k_ref, half_width), comet_refine_seeds,
 * comet_scan_rss of the new set, half_width *= shrink.  Then the k_final finally selected seeds
 * by the same rule with the last half_width, each classified (R28):
 *   final_seed  dev [n_part][k_final][6] (x,y,z,px,py,pz; NaN where none), final_rss dev [n_part][k_final],
 *   final_dca   dev [n_part][k_final][n_fired], cls dev [n_part][k_final][n_hits]
 *   part_off    HOST [n_part+1], part_off[0] = 0, part_off[n_part] = n_seeds, no empty partition
 *   work        dev, comet_stage_work_bytes(...) bytes
 *   z_run       the caller's knowledge about `seeds` as in comet_scan_rss (iteration 0 only)
 * Only enqueues work on cuda_stream (plus the ctx's internal streams, see comet_scan_rss). */
int comet_scan_stage(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                     int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                     const double* wire_a, const double* wire_b, int32_t n_wires,
                     const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                     int32_t n_fired, int32_t n_hits, double cutoff_cm,
                     const int64_t* part_off, int32_t n_part,
                     const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                     int32_t k_ref, int32_t k_final, void* work,
                     double* final_seed, double* final_rss, double* final_dca, uint8_t* cls,
                     void* cuda_stream);

/* ---- sequential stages with hit removal (readings R33-R34) -------------------- */

/* "The hits classified previously were excluded in the seed scanning; therefore, the number of
 * wires gets reduced whenever a track is fitted".  Input convention (R33): a measured
 * hit is the adjacent pair of ghost entries (2m, 2m+1), so n_hits and every hit_off[i] are even.
 * Entry j is removed when cls[j] or cls[j ^ 1] is set; a wire left without entries leaves the fired
 * list; the order of wires and entries is kept.
 *   cls          dev [n_hits] 0/1 (e.g. one row of comet_scan_stage's cls)
 *   orig_in      dev [n_hits] entry numbers carried along (NULL = 0, 1, 2, ...), orig_out dev [n_hits] or NULL
 *   fired_out    dev [n_fired], hit_off_out dev [n_fired+1], rho_out dev [n_hits]: the reduced list
 *   counts       dev [2]: its number of fired wires and of entries */
int comet_remove_hits(comet_ctx* ctx, const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                      int32_t n_fired, int32_t n_hits, const uint8_t* cls, const int32_t* orig_in,
                      int32_t* fired_out, int32_t* hit_off_out, double* rho_out, int32_t* orig_out,
                      int32_t* counts, void* cuda_stream);

/* Bytes of the device work buffer of comet_scan_turns (0 for invalid arguments). */
size_t comet_turns_work_bytes(int64_t max_partition_seeds, int32_t n_fired, int32_t n_hits, int32_t k_ref,
                              const int32_t* n_grid);

/* The stage loop of PAPER.md:256 without the fit between the stages (GENFIT2, out of scope): the
 * last turn partition first (descending partition index); each stage is comet_scan_stage on that
 * partition's seeds (k_final = 1) against the hits that are left, the hits its best seed classifies
 * are removed (comet_remove_hits) before the previous turn is scanned; the loop stops when fewer
 * than min_wires fired wires are left or max_tracks stages are done (paper: 30 and 5) (R34).
 *   turn_seed   dev [n_part][6], turn_rss dev [n_part]: the stage's best seed (NaN where no stage ran)
 *   turn_cls    dev [n_part][n_hits]: the hits given to each turn, in the event's own entry numbering
 *   done, wires_before  dev [n_part] int32: 1 where a stage ran; fired wires it started with (0 elsewhere)
 *   work        dev, comet_turns_work_bytes(largest partition, n_fired, n_hits, k_ref, n_grid)
 *   z_run       as in comet_scan_rss, used for the partitions that start on a run
 * Only enqueues work: no host read, no synchronisation (the paper's host loop reads the reduced list back after
 * every fit).  Every stage is launched for the event's own list sizes; the reduced list is padded back
 * to n_fired wires with wires that have no entries, Eq. (1) runs over the wires that are left (a device counter), and
 * once the stop rule has fired every kernel of the later stages returns at once.  With the workspace reserved
 * (comet_reserve_scan) the whole loop can be captured into a CUDA graph. */
int comet_scan_turns(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds, int32_t z_run,
                     int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                     const double* wire_a, const double* wire_b, int32_t n_wires,
                     const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                     int32_t n_fired, int32_t n_hits, double cutoff_cm,
                     const int64_t* part_off, int32_t n_part,
                     const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                     int32_t k_ref, int32_t min_wires, int32_t max_tracks, void* work,
                     double* turn_seed, double* turn_rss, uint8_t* turn_cls,
                     int32_t* done, int32_t* wires_before, void* cuda_stream);

/* ---- Hough-transform transverse seeding (Fig. 10; readings R35-R37) ------------ */

/* Bytes of the device work buffer of comet_hough_seeds (0 for n_events < 0). */
size_t comet_hough_work_bytes(int32_t n_events);

/* "The transverse components of (theta, p_x, p_y) were extracted by finding a circle that is the
 * transverse projection of a helical trajectory [...] the Hough transform was applied to the set of
 * transverse positions of the fired wires", for a batch of events in one launch.
 * R35: a wire's transverse position is the (x, y) of its midpoint.  R36: the circle passes through
 * the origin, so u = x/(x^2+y^2), v = y/(x^2+y^2) lie on the line u cos(phi) + v sin(phi) = rho with
 * rho = 1/(2R) and phi the azimuth of the circle's centre; every fired wire votes once per direction
 * phi_j in the bin floor((rho - rho_min) inv_drho) if that lies in [0, n_rho) (fp64, one IEEE
 * operation per operation written here; no trigonometric function is evaluated: the tables are
 * inputs); the peak is the bin of most votes, ties -> the lowest j n_rho + k.  R37: R = 1/(2 rho*)
 * with rho* = rho_min + (k + 0.5)/inv_drho, centre R (cos, sin); the seed points are the two
 * intersections with the cylinder r = r_seed_cm, p_T = kappa |B_z| R along the tangent in the
 * particle's sense of rotation; the entrance is the one where the track moves outwards.
 *   wire_a, wire_b   dev SoA [3][n_wires] endpoints (cm)
 *   fired_wire       dev [ev_off[n_events]] wire indices in [0, n_wires), the events one after the other
 *   ev_off           dev [n_events+1] non-decreasing offsets into fired_wire, ev_off[0] = 0; n_events <= 65535
 *   cos_tab, sin_tab dev [n_phi]; n_phi >= 1, 1 <= n_rho <= 32768, n_phi n_rho < 2^31, inv_drho > 0
 *   acc              dev [n_events][n_phi][n_rho] int32 votes, or NULL to skip writing them
 *   peak             dev [n_events][3] int32: votes, j, k of the peak ((0, 0, 0) without votes)
 *   circle           dev [n_events][11]: R, centre x, y, entrance (x, y, p_x, p_y), exit (x, y, p_x, p_y);
 *                    NaN without votes; entrance/exit NaN when the circle does not reach r_seed_cm
 *   work             dev, comet_hough_work_bytes(n_events)
 * Indices in fired_wire are not checked on the device.  No host synchronisation. */
int comet_hough_seeds(comet_ctx* ctx, const double* wire_a, const double* wire_b, int32_t n_wires,
                      const int32_t* fired_wire, const int32_t* ev_off, int32_t n_events,
                      const double* cos_tab, const double* sin_tab, int32_t n_phi,
                      double rho_min, double inv_drho, int32_t n_rho,
                      int32_t charge, double bz_tesla, double r_seed_cm, void* work,
                      int32_t* acc, int32_t* peak, double* circle, void* cuda_stream);

/* ---- half tracks (readings R38-R42) ------------------------------------- */

/* "The hits of the event were also grouped into two sets for each half track".
 * R39: the half tracks meet at the apex of the Hough circle, on the line from the origin through
 * its centre c.  With m the (x, y) of a wire's midpoint, d = (c_x m_y - c_y m_x)/R and s = +1 if
 * c_x e_y - c_y e_x > 0 else -1 (e the entrance point): the wire's entries belong to the entrance
 * half iff s d > -overlap_cm and to the exit half iff s d <= overlap_cm (fp64, one IEEE operation
 * per operation written here).  A NaN circle puts nothing in either set.
 *   circle   dev [11]: one row of comet_hough_seeds' output (R, centre, entrance, exit)
 *   in_ent, in_exit  dev [n_hits] 0/1 */
int comet_half_hit_masks(comet_ctx* ctx, const double* wire_a, const double* wire_b, int32_t n_wires,
                         const int32_t* fired_wire, const int32_t* hit_off, int32_t n_fired, int32_t n_hits,
                         const double* circle, double overlap_cm, uint8_t* in_ent, uint8_t* in_exit,
                         void* cuda_stream);

/* "by flipping the charge and momentum" (R38): out = (x, -p) of seeds SoA
 * [6][seed_stride] -> SoA [6][out_stride] (out may be seeds itself); the caller passes -charge to
 * the scan and scans against -rho (the reversed tangent swaps left and right). */
int comet_flip_seeds(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                     double* out, int64_t out_stride, void* cuda_stream);

/* "the seeds which have any missing layer without the hits were excluded".  R40:
 * with l_max the highest layer holding a classified hit of the seed, ok = 1 iff every layer
 * 0..l_max holds one and l_max + 1 >= min_layers; nothing classified gives 0.
 *   cls         dev [n_sel][n_hits] (e.g. comet_scan_stage's cls);  ok  dev [n_sel] 0/1
 *   wire_layer  dev [n_wires], values in [0, 64) (not checked on the device) */
int comet_layer_veto(comet_ctx* ctx, const uint8_t* cls, int32_t n_sel,
                     const int32_t* fired_wire, const int32_t* hit_off, int32_t n_fired, int32_t n_hits,
                     const int32_t* wire_layer, int32_t n_wires, int32_t min_layers, uint8_t* ok,
                     void* cuda_stream);

/* "The complete sets of classified hits were formed by combinatorially merging two half sets, one
 * of which is from each direction".  R41: pair (a, b) is valid iff ok_e[a] and
 * ok_x[b]; its complete set is the union of the two half sets in the event's entry numbering.
 *   cls_e  dev [k_e][h_e], orig_e dev [h_e] (entry of the half list -> entry of the event, < n_hits),
 *   ok_e   dev [k_e]; the same for the exit side (k_x, h_x); 1 <= k_e, k_x <= 65535
 *   valid  dev [k_e][k_x] 0/1, cls dev [k_e][k_x][n_hits] (zeros where not valid), n_cls dev [k_e][k_x] */
int comet_merge_half_sets(comet_ctx* ctx, const uint8_t* cls_e, const int32_t* orig_e, const uint8_t* ok_e,
                          int32_t k_e, int32_t h_e, const uint8_t* cls_x, const int32_t* orig_x,
                          const uint8_t* ok_x, int32_t k_x, int32_t h_x, int32_t n_hits,
                          uint8_t* valid, uint8_t* cls, int32_t* n_cls, void* cuda_stream);

/* Bytes of the device work buffer of comet_scan_half_tracks (0 for invalid arguments). */
size_t comet_half_work_bytes(int64_t n_seeds_ent, int64_t n_seeds_exit, int32_t n_fired, int32_t n_hits,
                             int32_t k_ref, int32_t k_final, const int32_t* n_grid);

/* One turn partition as two half tracks (R38-R42): comet_half_hit_masks +
 * comet_remove_hits give the two hit lists; the entrance-side seeds are scanned forwards against
 * the entrance list and the exit-side seeds backwards (comet_flip_seeds, -charge, -rho) against
 * the exit list, each by comet_scan_stage with one partition and k_final finally selected seeds
 * (paper: 10 per side); comet_layer_veto; comet_merge_half_sets.  A half track ends at the apex:
 * pass r_stop_cm beyond the chamber (e.g. 1e3; R42).
 *   seeds_ent  dev SoA [6][n_ent], seeds_exit dev SoA [6][n_exit] (physical momenta), n_* >= 1
 *   circle     dev [11] (comet_hough_seeds); wire_layer dev [n_wires]; n_hits and every hit_off even (R33)
 *   half_seed  dev [2][k_final][6]: the finally selected seeds, entrance side then exit side (physical
 *              momenta; NaN where none); half_rss dev [2][k_final]; half_ok dev [2][k_final]
 *   half_cls   dev [2][k_final * n_hits]: side h's rows are [k_final][counts_host[2 h + 1]] (dense), entries
 *              in the numbering of its half list; half_orig dev [2][n_hits]: half-list entry -> event entry
 *   counts_host  HOST [4]: fired wires and entries of the entrance list, then of the exit list
 *   valid dev [k_final][k_final], cls dev [k_final][k_final][n_hits], n_cls dev [k_final][k_final]
 *   work       dev, comet_half_work_bytes(n_ent, n_exit, n_fired, n_hits, k_ref, k_final, n_grid)
 * Synchronises cuda_stream once (the sizes of the two hit lists set the launches of the scans). */
int comet_scan_half_tracks(comet_ctx* ctx, const double* seeds_ent, int64_t n_ent,
                           const double* seeds_exit, int64_t n_exit,
                           int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                           const double* wire_a, const double* wire_b, int32_t n_wires,
                           const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                           int32_t n_fired, int32_t n_hits, double cutoff_cm,
                           const int32_t* wire_layer, const double* circle, double overlap_cm, int32_t min_layers,
                           const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                           int32_t k_ref, int32_t k_final, void* work,
                           double* half_seed, double* half_rss, uint8_t* half_ok, uint8_t* half_cls,
                           int32_t* half_orig, int32_t* counts_host,
                           uint8_t* valid, uint8_t* cls, int32_t* n_cls, void* cuda_stream);

/* Bytes of the device work buffer of comet_scan_turns_half (0 for invalid arguments). */
size_t comet_turns_half_work_bytes(int64_t max_seeds_ent, int64_t max_seeds_exit, int32_t n_fired, int32_t n_hits,
                                   int32_t k_ref, int32_t k_final, const int32_t* n_grid);

/* The event loop of Fig. 13 with half tracks and without the fits (GENFIT2, out of
 * scope): the last turn partition first; comet_scan_half_tracks of the turn's entrance- and
 * exit-side seed sets against the hits that are left; the complete set that goes on is the valid
 * pair with the most classified entries, ties -> the lowest a k_final + b (R43: stands in for the
 * highest NDF of the fits); its hits are removed (comet_remove_hits) before the
 * previous turn.  Stops when fewer than min_wires fired wires are left, max_tracks turns are done
 * (R34) or a turn has no valid pair.  The circle is the same for every turn (:256).
 *   seeds_ent   dev SoA [6][n_ent], off_ent HOST [n_part+1] (off[0] = 0, off[n_part] = n_ent, no empty
 *               partition); the same for the exit side
 *   turn_pair   dev [n_part][2] int32 (a, b), -1 where no turn was taken; turn_n dev [n_part] its entries
 *   turn_seed   dev [n_part][2][6]: the pair's entrance- and exit-side seeds (NaN where none)
 *   turn_cls    dev [n_part][n_hits]: the turn's complete set in the event's own entry numbering
 *   done_host, wires_before_host  HOST [n_part]: 1 where a turn was taken; fired wires its scan started with
 *   work        dev, comet_turns_half_work_bytes(largest entrance set, largest exit set, n_fired, n_hits, ...)
 * Synchronises cuda_stream twice per turn (the sizes of the hit lists set the launches). */
int comet_scan_turns_half(comet_ctx* ctx, const double* seeds_ent, const int64_t* off_ent, int64_t n_ent,
                          const double* seeds_exit, const int64_t* off_exit, int64_t n_exit, int32_t n_part,
                          int32_t charge, double bz_tesla, double step_cm, int32_t n_steps, double r_stop_cm,
                          const double* wire_a, const double* wire_b, int32_t n_wires,
                          const int32_t* fired_wire, const int32_t* hit_off, const double* rho,
                          int32_t n_fired, int32_t n_hits, double cutoff_cm,
                          const int32_t* wire_layer, const double* circle, double overlap_cm, int32_t min_layers,
                          const double* half_width, const int32_t* n_grid, int32_t n_iter, double shrink,
                          int32_t k_ref, int32_t k_final, int32_t min_wires, int32_t max_tracks, void* work,
                          int32_t* turn_pair, int32_t* turn_n, double* turn_seed, uint8_t* turn_cls,
                          int32_t* done_host, int32_t* wires_before_host, void* cuda_stream);

/* ---- seed grids as inputs (readings R17, R44) --------------------------------- */

/* "A seed set was prepared by combining each component from the grids of the ranges":
 * the first-iteration seed set of n_part turn partitions built on the device from its axes instead of
 * 6 x S doubles crossing the bus.  axes is [n_part][A] doubles, A = comet_grid_axes_len(...) =
 * 2 + n_p + 2 n_ct + 2 n_phi + n_z, per partition:
 *   x, y (the seed point on the r = 50 cm cylinder) | |p| [n_p] | sin(theta) [n_ct] |
 *   cos(theta) [n_ct] | cos(phi0) [n_phi] | sin(phi0) [n_phi] | z0 [n_z]
 * (tables: no transcendental function is evaluated by the library).  Seed ((i_p n_ct + i_ct) n_phi +
 * i_phi) n_z + i_z of partition q, at index q G + that, G = n_p n_ct n_phi n_z (R17), is
 *   (x, y, z0[i_z], (|p| sin) cos(phi0), (|p| sin) sin(phi0), |p| cos(theta))
 * each product one IEEE multiplication in the order written (R44).
 *   axes    dev [n_part][A];  seeds  dev SoA [6][seed_stride], seed_stride >= n_part G, written
 * z is the fastest index, so comet_grid_z_run(n_z) -- the largest power of two <= 32 dividing n_z -- is a
 * valid z_run promise for scans of this set (and of any partition of it). */
int comet_seed_grid(comet_ctx* ctx, const double* axes, int32_t n_part, int32_t n_p, int32_t n_ct,
                    int32_t n_phi, int32_t n_z, double* seeds, int64_t seed_stride, void* cuda_stream);
size_t comet_grid_axes_len(int32_t n_p, int32_t n_ct, int32_t n_phi, int32_t n_z);   /* 0 for invalid shapes */
int32_t comet_grid_z_run(int32_t n_z);

/* The z_run of an arbitrary seed set: the largest power of two r <= 32 such that every aligned run of r
 * consecutive seeds is bit-identical in (x, y, p_x, p_y, p_z), written to *z_run_host (HOST).  One small
 * kernel; synchronises cuda_stream (a query made once per seed set, not in the hot loop). */
int comet_seed_runs(comet_ctx* ctx, const double* seeds, int64_t seed_stride, int64_t n_seeds,
                    int32_t* z_run_host, void* cuda_stream);

/* Keeps a copy of the detector's wire endpoints (HOST SoA [3][n_wires] each) on the device for the host-buffer
 * entry points below (the geometry is a constant of the detector, not an input of an event).  Synchronises
 * cuda_stream; n_wires = 0 frees the copy.  comet_get_geometry returns the device pointers (NULL when none). */
int comet_set_geometry(comet_ctx* ctx, const double* wire_a_host, const double* wire_b_host, int32_t n_wires,
                       void* cuda_stream);
int comet_get_geometry(const comet_ctx* ctx, const double** wire_a_dev, const double** wire_b_dev, int32_t* n_wires);

/* ---- whole event from host buffers ------------------------------------------------------- */

/* Runs A, B and C for one event whose inputs and outputs live in HOST memory (pinned memory makes
 * the copies asynchronous): copies the inputs to the device, runs comet_scan_rss (track on chip) when
 * track_budget_bytes == 0 -- the seeds are then uploaded sub-slab by sub-slab on the ctx's internal
 * streams, so the upload overlaps the kernels of the sub-slabs already on the device --, else comet_seed_extrapolate + comet_dca_rss over slabs of seeds that fit
 * `track_budget_bytes` of track workspace (grown inside the ctx when needed), copies
 * best_seed/best_rss/best_dca/cls (and rss if rss_host != NULL) back and synchronises the stream.
 * All array arguments have the shapes of the device-buffer calls above.  wire_a_host = wire_b_host = NULL
 * uses the geometry of comet_set_geometry (n_wires is then ignored). */
int comet_scan_event_host(comet_ctx* ctx, const double* seeds_host, int64_t n_seeds,
                          int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                          double r_stop_cm,
                          const double* wire_a_host, const double* wire_b_host, int32_t n_wires,
                          const int32_t* fired_wire_host, const int32_t* hit_off_host,
                          const double* rho_host, int32_t n_fired, int32_t n_hits, double cutoff_cm,
                          const int64_t* part_off_host, int32_t n_part, size_t track_budget_bytes,
                          int64_t* best_seed_host, double* best_rss_host, double* best_dca_host,
                          uint8_t* cls_host, double* rss_host, void* cuda_stream);

/* The same event with its seed sets given as grid axes (comet_seed_grid; HOST [n_part][A]) and the geometry
 * of comet_set_geometry: per event only the axes, the fired wires and the hit entries cross the bus (a few
 * KB).  Copies them in (one transfer, through a pinned staging buffer of the ctx: the caller's arrays need not
 * be pinned), builds the seeds on the device, runs comet_scan_rss with z_run = comet_grid_z_run(n_z) and
 * comet_select_and_classify with part_off[q] = q G, copies best_seed / best_rss / best_dca / cls back (one
 * transfer; rss [n_part G] too if rss_host != NULL) and synchronises the stream. */
int comet_scan_event_grid_host(comet_ctx* ctx, const double* axes_host, int32_t n_part, int32_t n_p,
                               int32_t n_ct, int32_t n_phi, int32_t n_z,
                               int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                               double r_stop_cm,
                               const int32_t* fired_wire_host, const int32_t* hit_off_host,
                               const double* rho_host, int32_t n_fired, int32_t n_hits, double cutoff_cm,
                               int64_t* best_seed_host, double* best_rss_host, double* best_dca_host,
                               uint8_t* cls_host, double* rss_host, void* cuda_stream);

/* The same call in two halves, for a stream of events: comet_scan_event_grid_submit copies the inputs into the
 * staging buffer of `slot` (0 <= slot < COMET_EVENT_SLOTS) and enqueues the upload, the seed grid, steps A-C and the
 * download of the results on `cuda_stream`; it returns without waiting.  comet_scan_event_grid_collect waits for
 * that event's results and copies them to the caller's arrays.  With two slots the host side of event k + 1
 * (packing, upload, launches) overlaps the kernels of event k; the events of one ctx run one after the other on
 * the device (they share the scan workspace), so all submits of a ctx go to the same stream.
 * A slot holds one event at a time: COMET_EINVAL for a submit into a slot that has not been collected, or a
 * collect from an empty one.  The caller's input arrays may be reused as soon as submit returns. */
#define COMET_EVENT_SLOTS 2
int comet_scan_event_grid_submit(comet_ctx* ctx, int32_t slot, const double* axes_host, int32_t n_part, int32_t n_p,
                                 int32_t n_ct, int32_t n_phi, int32_t n_z,
                                 int32_t charge, double bz_tesla, double step_cm, int32_t n_steps,
                                 double r_stop_cm,
                                 const int32_t* fired_wire_host, const int32_t* hit_off_host,
                                 const double* rho_host, int32_t n_fired, int32_t n_hits, double cutoff_cm,
                                 void* cuda_stream);
int comet_scan_event_grid_collect(comet_ctx* ctx, int32_t slot, int64_t* best_seed_host, double* best_rss_host,
                                  double* best_dca_host, uint8_t* cls_host);

/* ---- an entry point that allocates nothing ---------------------------------------------------- */

/* The per-partition argmin of step C (reading R15) on its own, for callers that cannot call cudaMalloc
 * (code under CUDA-graph capture, tight serving loops, harnesses that forbid it): no ctx -- comet_create
 * allocates --, no cudaMalloc / cudaFree / allocating routine, on the CURRENT device and `cuda_stream`.
 * best_seed[p] = lowest-index argmin of rss over [part_off[p], part_off[p + 1]) (-1 for an empty partition),
 * best_rss[p] its value (NaN for an empty partition); the NaN rule is comet_select_and_classify's, and the
 * results are the same numbers as that call's best_seed / best_rss.
 *   rss        dev [n_seeds]            part_off  HOST [n_part + 1], non-decreasing, within [0, n_seeds]; read before returning
 *   best_seed  dev [n_part] (written)   best_rss  dev [n_part] (written); both owned by the caller
 * The partial minima of the two-stage search (64 slices per partition) live in a file-scope device array of
 * COMET_STATIC_MAX_PART x 64 x 16 bytes = 64 KB that every GPU that loads the library holds until the process
 * exits.  n_part > COMET_STATIC_MAX_PART: COMET_ELIMIT, nothing is launched; n_seeds has no limit.
 * ALL calls on a device share that array: calls whose kernels can overlap on the GPU (different streams
 * without an ordering between them) race and give undefined results -- order them.  The array keeps the last
 * call's contents; every slot a call reads it has written itself first, so nothing needs clearing between calls.
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress); make that call
 * outside a stream capture.  COMET_ECUDA if the address cannot be resolved or a launch fails. */
#define COMET_STATIC_MAX_PART 64
int comet_argmin_static(const double* rss, int64_t n_seeds, const int64_t* part_off, int32_t n_part,
                        int64_t* best_seed, double* best_rss, void* cuda_stream);

/* ---- measurement helper ------------------------------------------------------------------ */

/* Enqueues a dependent-free DFMA loop on every SM (`iters` FMAs per thread on 8 chains) and
 * returns the number of FP64 FMA instructions it executes per launch in *n_fma (host).  Timing it
 * with CUDA events gives the FP64 pipe peak of the device the roofline is quoted against. */
int comet_fp64_peak_probe(comet_ctx* ctx, int32_t iters, double* sink_dev, double* n_fma,
                          void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* COMET_H_ */
