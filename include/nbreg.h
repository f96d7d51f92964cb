/*
 * nbreg.h -- C ABI of libnbreg: the GPU regular-force step of the fourth-order Hermite /
 * Ahmad-Cohen neighbour scheme (arXiv 1504.03687, "NBODY6++GPU"), B200 / sm_100a only.
 *
 * For a block of active i-particles the library predicts all N j-particles to the block time and
 * sums, over every j, the Newtonian acceleration, its time derivative (jerk) and the potential;
 * pairs inside particle i's neighbour radius are excluded from the sums and emitted as i's
 * neighbour list (section 2; section 3.2.1; section 3.3.3; Table 1).
 *
 * Conventions
 *   - G = 1 (N-body units).  All floating-point arguments are FP64.
 *   - Arrays of vectors are [n][3] row-major.  Indices are 0-based int32.
 *   - "DEVICE" pointers are CUDA device pointers valid on the current device; "HOST" pointers are
 *     ordinary (pageable or pinned) host memory.  The caller owns every pointer it passes; the
 *     library copies what it needs and never retains a caller pointer after the call returns
 *     (for DEVICE variants: after the work enqueued by the call has run).
 *   - DEVICE variants enqueue on the context's stream (nb_set_stream; default: the legacy default
 *     stream) and return without synchronising.  Outputs are valid once the caller has synchronised
 *     that stream (or called nb_synchronize).  HOST variants return after their results are in the
 *     caller's host buffers.
 *   - Every call returns an int status: NB_OK or one of the NB_E* codes; nb_strerror() names it.
 *     No exceptions, no aborts, no output on stdout/stderr.  A CUDA failure is sticky: every later
 *     call on that context returns NB_ECUDA.  Neighbour-list overflow is NOT an error.
 *   - There is no CPU fallback: without a usable sm_100 device nb_open fails with NB_ECUDA.
 *   - Results are bitwise reproducible run to run for fixed inputs and a fixed launch plan (two-stage
 *     fixed-order reduction, no floating-point atomics); list rows are sorted, so they are too, except
 *     WHICH nb_cap neighbours an overflowed row keeps.
 *
 * Precision of the pair arithmetic (the paper does not state its kernel's precision; DESIGN.md
 * "Precision"): positions are differenced at FP64-equivalent accuracy -- as two-float hi/lo pairs (2^-48
 * relative), or, for a warp whose 64 active particles lie within G = 8 neighbour radii of their common
 * centre, in that warp's own FP32 frame (relative error of a difference <= 1.8e-7 + 2.4e-7 G at the
 * neighbour boundary, translation invariant) --, velocities and masses are rounded to FP32, the pair terms
 * are FP32 with an SFU reciprocal square root, sums are FP32 within a j-tile and FP64 across tiles.
 * Guaranteed against the FP64 definition: acceleration max rel 1e-5 / rms 1e-6, jerk 1e-4 / 1e-5,
 * potential 1e-6; neighbour sets identical except pairs with |r^2 - h^2| / h^2 < 1e-5.
 * Velocity frame: v is kept as ONE FP32, so a bulk velocity common to all bodies enters the jerk with a
 * relative error of about 6e-8 |v_bulk| / sigma (sigma = velocity dispersion): the jerk bounds hold for
 * |v_bulk| <~ 100 sigma.  Integrate a cluster on a galactic orbit in its own frame.
 */
#ifndef NBREG_H
#define NBREG_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nb_ctx nb_ctx; /* opaque; owns all internal device memory */

enum {
    NB_OK = 0,
    NB_EINVAL = 1, /* null pointer, N <= 0, nb_cap <= 0, n_i < 0 or n_i > N, unknown key            */
    NB_ESTATE = 2, /* nb_predict_all before nb_set_j, nb_regular before nb_predict_all; also: the
                      current CUDA device is not the one the context was opened on                 */
    NB_ENOMEM = 3, /* device (or staging) allocation failed                                        */
    NB_ECUDA = 4,  /* CUDA error (sticky); nb_last_cuda_error() returns the cudaError_t            */
    NB_EOVERFLOW = 5, /* two-level AC stepping only: a neighbour list overflowed nb_cap (not sticky) */
    NB_ELIMIT = 6  /* nb_next_block_static only: N is larger than NB_STATIC_MAX_N                    */
};

/* Create a context for N j-particles and a neighbour-list capacity of nb_cap entries per active
 * particle (north_star: nb_open(N); the capacity has to come from somewhere -- DESIGN.md R18).
 * Allocates: the FP64 j-state (14 N doubles), predicted records (40 B per particle, padded), counters,
 * split-j scratch (grown on demand); a second, 128 B/body gather copy of the state only when the first
 * nb_irregular / nb_correct call asks for it. */
int nb_open(int64_t N, int32_t nb_cap, nb_ctx **out);
int nb_close(nb_ctx *ctx);

/* cudaStream_t (as void*) on which all later calls enqueue. NULL = legacy default stream. */
int nb_set_stream(nb_ctx *ctx, void *cuda_stream);
int nb_synchronize(nb_ctx *ctx);

/* a1 "Send.R" (Table 1): ingest the state of ALL N particles at their own times t0[j]:
 * m[N], x0[N][3], v0[N][3], a0[N][3] (total acceleration at t0), j0[N][3] (total jerk at t0),
 * t0[N].  The library re-lays the data out (AoS -> SoA) into its own copy.  DEVICE pointers. */
int nb_set_j(nb_ctx *ctx, const double *m, const double *x0, const double *v0, const double *a0,
             const double *j0, const double *t0);
/* Same with HOST pointers: host->device copies, then the same re-layout kernel. */
int nb_set_j_host(nb_ctx *ctx, const double *m, const double *x0, const double *v0,
                  const double *a0, const double *j0, const double *t0);

/* Incremental "Send.R": after a block step only the n integrated
 * particles changed -- replace the state of bodies idx[0..n) (unique, in range, unchecked) by
 * m[n], x0[n][3], v0[n][3], a0[n][3], j0[n][3], t0[n].  The predicted records become stale:
 * nb_regular needs a new nb_predict_all.  DEVICE pointers.  Requires nb_set_j; n = 0 is a no-op. */
int nb_update_j(nb_ctx *ctx, int32_t n, const int32_t *idx, const double *m, const double *x0,
                const double *v0, const double *a0, const double *j0, const double *t0);

/* a2 "Pred." (Table 1): predict every particle to time t,
 *     dt = t - t0[j];  xp = x0 + v0 dt + a0 dt^2/2 + j0 dt^3/6;  vp = v0 + a0 dt + j0 dt^2/2
 * in FP64, and store the predicted record the force kernel reads (x as hi/lo FP32 pair, v and m
 * as FP32).  Any t (also t < t0[j]) is allowed.  Requires nb_set_j.
 * The predictor kernel itself is launched by the first call that reads the records (NB_TUNE_FUSE_PREDICT):
 * a block of <= 128 active particles predicts inside its force kernel instead -- same arithmetic, same
 * records, results independent of which route was taken up to the summation order. */
int nb_predict_all(nb_ctx *ctx, double t);

/* Test/inspection hook: the predicted state exactly as the force kernel sees it, widened to FP64:
 * xp[N][3] = (double)hi + (double)lo, vp[N][3] = (double)v_fp32.  DEVICE pointers. */
int nb_get_predicted(nb_ctx *ctx, double *xp, double *vp);

/* a3-a7 "Reg." (Table 1): for k = 0..n_i-1, i = idx_i[k]:
 *     over all j != i (by index) at the predicted positions/velocities, r = x_j - x_i, v = v_j - v_i:
 *       r^2 <  h2_i[k] : j is a neighbour of i -- listed, excluded from the sums
 *       r^2 >= h2_i[k] : acc[k]  += m_j r / r^3
 *                        jerk[k] += m_j ( v / r^3 - 3 (r.v) r / r^5 )
 *                        pot[k]  -= m_j / r
 *   nnb[k]      = TRUE number of neighbours (may exceed nb_cap)
 *   overflow[k] = nnb[k] > nb_cap
 *   nblist[k][0 .. min(nnb[k], nb_cap))  = neighbour indices j in ascending order (rows are sorted
 *                 after the pass whenever nb_cap <= 32768; above that the order is unspecified); on
 *                 overflow any nb_cap of the true neighbours.  Entries beyond that are left untouched.
 *   The sums exclude ALL true neighbours whether or not the list overflowed.
 * h2_i[k] <= 0 means "no neighbours" (total force / full potential).  The i-particle's own state is
 * its predicted record (index idx_i[k]); the self pair is skipped by index.
 * idx_i must be unique and in [0, N) (unchecked).  n_i = 0 is a valid no-op.
 * Shapes: idx_i[n_i] int32, h2_i[n_i], acc[n_i][3], jerk[n_i][3], pot[n_i], nnb[n_i] int32,
 * nblist[n_i][nb_cap] int32, overflow[n_i] int32.  DEVICE pointers.  Requires nb_predict_all. */
int nb_regular(nb_ctx *ctx, int32_t n_i, const int32_t *idx_i, const double *h2_i, double *acc,
               double *jerk, double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow);
/* Full-N pass (section 3.3.2: forces and neighbour lists of ALL particles are initialised with
 * the same GPU kernel; the same pass with h2 = 0 gives every particle's full potential
 * for the energy check): nb_regular with the identity block idx_i[k] = k, n_i = N.
 * Shapes as nb_regular with n_i = N: h2[N], acc[N][3], jerk[N][3], pot[N], nnb[N], overflow[N],
 * nblist[N][nb_cap] -- or nblist = NULL: neighbours are counted (nnb, overflow exact) but not stored
 * (N x nb_cap x 4 B is 2 GiB at N = 1M, cap = 512).  DEVICE pointers.  Requires nb_predict_all. */
int nb_regular_all(nb_ctx *ctx, const double *h2, double *acc, double *jerk, double *pot,
                   int32_t *nnb, int32_t *nblist, int32_t *overflow);
/* Same as nb_regular with HOST pointers: copies idx_i/h2_i in, runs, copies all outputs back, synchronises.
 * nblist may be NULL to skip the list copy-back (the list is still built on the device). */
int nb_regular_host(nb_ctx *ctx, int32_t n_i, const int32_t *idx_i, const double *h2_i, double *acc,
                    double *jerk, double *pot, int32_t *nnb, int32_t *nblist, int32_t *overflow);

/* One whole block step a1-a7 through HOST buffers, pipelined: equivalent to
 *     nb_set_j_host(m .. t0);  nb_predict_all(t);  nb_regular_host(n_i .. overflow)
 * (Table 1: Send.R, Pred., Reg. of one regular block), but the j-state is sent in chunks
 * (1/16, 1/16, 1/8, 1/4, 1/2 of the bodies) on a second stream, each chunk is re-laid out and
 * predicted as it lands, and the force kernel runs chunk by chunk behind the copies, so that only
 * the first chunk's transfer is exposed.  The active particles' own records (a3) come from their
 * state gathered on the host (14 doubles each) and predicted with the same arithmetic, so they are
 * bitwise the records of bodies idx_i[k].  Results equal those of the three separate calls except
 * for the order in which the per-chunk partial sums are added (FP64, fixed and reproducible); neighbour
 * lists, counts and flags are identical.  Leaves the context as after set_j + predict_all(t).
 * idx_i is range-checked here (NB_EINVAL).  HOST pointers (pinned memory makes the copies
 * asynchronous); nblist may be NULL to skip the list copy-back.  Returns with the results in place. */
int nb_step_host(nb_ctx *ctx, const double *m, const double *x0, const double *v0, const double *a0,
                 const double *j0, const double *t0, double t, int32_t n_i, const int32_t *idx_i,
                 const double *h2_i, double *acc, double *jerk, double *pot, int32_t *nnb,
                 int32_t *nblist, int32_t *overflow);

/* Neighbour ("irregular") force on the GPU ("the irregular force
 * accumulates only the neighbor forces"; "predict all neighbors and do the force calculation
 * within one loop"; the paper runs this step on AVX/SSE CPUs).  For k = 0..n_i-1, i = idx_i[k]:
 * particle i and each j in nblist[k][0 .. min(nnb[k], nb_cap)) are predicted to time t from the FP64
 * j-state (same polynomial as nb_predict_all; nb_predict_all itself is NOT required) and
 *     acc[k] = sum_j m_j r / r^3,  jerk[k] = sum_j m_j ( v / r^3 - 3 (r.v) r / r^5 ),
 *     pot[k] = - sum_j m_j / r           (pot may be NULL)
 * in FP64 throughout (max rel. error vs the FP64 definition ~1e-13).  nnb / nblist have the layout
 * nb_regular writes ([n_i], [n_i][nb_cap]) and may be its outputs unchanged; a row that overflowed
 * contributes its nb_cap stored entries.  A large block (NB_TUNE_IRR_PRED_MIN bodies or more) predicts all N bodies
 * once into library-owned 64 B records and gathers those; the results are the same bits.  DEVICE pointers.
 * Requires nb_set_j. */
int nb_irregular(nb_ctx *ctx, double t, int32_t n_i, const int32_t *idx_i, const int32_t *nnb,
                 const int32_t *nblist, double *acc, double *jerk, double *pot);

/* ---- The steps either side of the regular-force pass: block time steps, active
 * selection, Hermite corrector.  The paper prints none of these formulas; they are the textbook
 * fourth-order Hermite scheme with hierarchical block steps that it names (Makino 1991,
 * Makino & Aarseth 1992) -- DESIGN.md readings R27-R31.  All pointers DEVICE unless marked HOST. */

/* Block time steps dt[N] (each an integer power of 0.5 with t0[j] a multiple of dt[j]; unchecked).
 * Copied.  Requires nb_set_j. */
int nb_set_steps(nb_ctx *ctx, const double *dt);
/* Start-up steps from the stored a0, j0: dt_j = largest power of 0.5 <= min(eta_s |a0| / |j0|, dt_max),
 * clipped below at dt_max 2^-40; |a0| = |j0| = 0 gives dt_max (reading R32). */
int nb_init_steps(nb_ctx *ctx, double eta_s, double dt_max);

/* Active selection for the next block ("active particles ... are integrated together"; P:89
 * section 3.3.1, Figures 1-2): t_next = min_j (t0_j + dt_j) and the bodies with t0_j + dt_j == t_next,
 * ascending, into idx_act (DEVICE, room for N).  *t_next and *n_act are HOST outputs: the call
 * synchronises the stream.  (The paper's step-sorted list exists so that a CPU never scans N bodies;
 * here the scan is 16 B/body of HBM traffic, ~3 us at N = 1M, and the list is not kept.) */
int nb_next_block(nb_ctx *ctx, double *t_next, int32_t *n_act, int32_t *idx_act);

/* Hermite corrector and new block step for the n active bodies idx[0..n) whose new acceleration
 * acc1[n][3] and jerk jerk1[n][3] were evaluated at time t = t0 + dt at the predicted state (the total
 * force: nb_regular with h2 = 0, or nb_regular + nb_irregular added by the caller).  With h = dt:
 *     a2 = ( -6 (a0 - a1) - h (4 j0 + 2 j1) ) / h^2       a3 = ( 12 (a0 - a1) + 6 h (j0 + j1) ) / h^3
 *     x1 = x0 + v0 h + a0 h^2/2 + j0 h^3/6 + a2 h^4/24 + a3 h^5/120
 *     v1 = v0 + a0 h + j0 h^2/2 + a2 h^3/6 + a3 h^4/24
 *     dt_req = sqrt( eta (|a1| |a2'| + |j1|^2) / (|j1| |a3| + |a2'|^2) ),  a2' = a2 + h a3
 *     new step: 2 dt if dt_req >= 2 dt, 2 dt <= dt_max and t is a multiple of 2 dt; else dt halved
 *     while it exceeds dt_req, but never below dt_max 2^-40; dt_req = 0 or NaN keeps the step (reading R32).
 * The stored state of these bodies becomes (x1, v1, a1, j1, t0 = t, new step); the predicted records
 * become stale (nb_regular needs a new nb_predict_all).  FP64.  idx unique, in range, unchecked. */
int nb_correct(nb_ctx *ctx, double t, int32_t n, const int32_t *idx, const double *acc1,
               const double *jerk1, double eta, double dt_max);

/* One whole block step in ONE call (SURVEY 8(f) NEXT-3 "device-side block loop"; P:47 block steps, P:89 the
 * cost of selection against small deep blocks, P:45 corrector):
 *     selection  t_next = min_j (t0_j + dt_j), active = {j : t0_j + dt_j = t_next} ascending (two launches: a
 *                minimum pass and a count / look-back prefix / ordered scatter pass; the block descriptor
 *                {t_next, n, status} is stored straight into mapped host memory -- the only host read of the step)
 *  -> prediction to t_next + regular force of the active block (a2-a7; blocks of <= 128 particles predict
 *                inside the force kernel)
 *  -> if h2_all != NULL: the neighbour force on the lists just written, added in place
 *  -> nb_correct for the block (corrector, Aarseth step, block rule; reading R31: one total force per body).
 * h2_all: DEVICE [N] squared neighbour radii indexed by BODY, or NULL: no neighbours (the regular pass gives
 * the total force, no lists are built).  If t_next > t_stop nothing is integrated: *n_act = 0, the state is
 * untouched (use t_stop = the end of the run; DBL_MAX never stops).  HOST outputs *t_next, *n_act.  Small
 * blocks are enqueued speculatively (NB_TUNE_SPECULATE), so the GPU does not wait for the host.  The block's
 * results stay in library-owned DEVICE buffers until the next nb_block_step (nb_get_block copies them out).  The kernels
 * after the selection are enqueued without a further synchronisation.  Requires nb_set_j and steps. */
int nb_block_step(nb_ctx *ctx, const double *h2_all, double eta, double dt_max, double t_stop,
                  double *t_next, int32_t *n_act);
/* Copy the last block's results into the caller's DEVICE buffers (any may be NULL), each with room for n_cap rows:
 * idx_act[n], acc[n][3], jerk[n][3], pot[n] -- the TOTAL force handed to the corrector --, nnb[n],
 * nblist[n][nb_cap] (NB_ESTATE if the step ran without h2_all), overflow[n], where n = min(n_cap, size of the last
 * block).  That size is the *n_act nb_block_step returned; after nb_run_blocks ask NB_INFO_LAST_BLOCK_N.  NB_ESTATE if
 * the last block loop was nb_ac_step / nb_ac_run (their results: nb_ac_get).  Enqueued on the stream. */
int nb_get_block(nb_ctx *ctx, int32_t n_cap, int32_t *idx_act, double *acc, double *jerk, double *pot, int32_t *nnb,
                 int32_t *nblist, int32_t *overflow);

/* ---- Two-level Ahmad-Cohen stepping ("the full force of one particle is separated
 * into two parts: regular and irregular forces ... there are regular (large) time steps and irregular (small)
 * time steps ... During the irregular step, the regular force and its first order derivative calculated at the
 * last regular step are used for the particle position and velocity prediction"; P:215 and Table A1: eta_I,
 * eta_R).  The paper prints no formulas: DESIGN.md readings R33-R38 (the Hermite AC scheme of Makino & Aarseth
 * 1992).  The library keeps per body the irregular force aI, jI (at its last irregular time, over its list), the
 * regular force aR, jR (at its last regular time tR), the steps dtI <= dtR and its neighbour list; the j-state
 * read by the predictor holds the TOTAL a0 = aI + aR + jR (t0 - tR), j0 = jI + jR.
 *
 * nb_ac_init: after nb_set_j with every t0[j] = t_start (a0, j0 are ignored and overwritten): full regular pass
 * with the radii h2_all[N] (DEVICE, copied; squared, indexed by body) -> aR, jR and every list; neighbour force
 * over the lists -> aI, jI; start-up steps dtR = initial step of the regular force, dtI = min(initial step of the
 * irregular force, dtR), dtI = dtR for a body without neighbours.  *n_overflow (HOST, may be NULL) = number of
 * lists longer than nb_cap; if any, returns NB_EOVERFLOW and AC stepping stays unavailable (shrink the radii:
 * radius control is the caller's, reading R38).  Allocates 6 N vectors + N x nb_cap list entries.
 * NB_ESTATE if some t0[j] != t_start (checked on the device): this is a START-UP call, not a way to re-list a
 * cluster in mid-run -- for that see nb_ac_set_radii.
 * Any call that replaces or advances the state outside the two-level scheme (nb_set_j, nb_set_j_host,
 * nb_step_host, nb_update_j, nb_set_steps, nb_init_steps, nb_correct, nb_block_step, nb_run_blocks) ends it:
 * nb_ac_step then returns NB_ESTATE until the next nb_ac_init. */
int nb_ac_init(nb_ctx *ctx, double t_start, const double *h2_all, double eta_s, double dt_max,
               int32_t *n_overflow);
/* One block of the two-level scheme: t_next = min_j (t0_j + dtI_j); the bodies due then take an IRREGULAR step
 * (neighbour force over their lists at the predicted state, regular force extrapolated linearly, Hermite corrector
 * over dtI, new dtI with eta_I, never above dtR); those whose regular step is due as well (tR + dtR = t_next)
 * take a REGULAR step too: regular force with new lists (nb_regular of that sub-block, prediction fused for small
 * ones), neighbour force over the new lists, regular force w.r.t. the old list = total - irregular(old), the regular
 * correction a2R dtR^4/24 + a3R dtR^5/120 (v: dtR^3/6, dtR^4/24) added to the corrected state, both polynomials
 * restarted from the new list, new dtR with eta_R.  HOST outputs *t_next, *n_irr (all active bodies), *n_reg.
 * If t_next > t_stop nothing happens (*n_irr = 0).  If a new list overflows, NB_EOVERFLOW is returned BEFORE
 * anything is corrected (*n_reg = number of overflowed rows; the state is untouched).  Blocks without a regular
 * step cost O(n_irr x neighbours), not O(N).  One host read-back per block (two when regular steps are due). */
int nb_ac_step(nb_ctx *ctx, double eta_I, double eta_R, double dt_max, double t_stop, double *t_next,
               int32_t *n_irr, int32_t *n_reg);
/* The block loop itself (SURVEY 8(f) NEXT-3 "device-side block loop"): nb_ac_step / nb_block_step repeated inside
 * the library until nothing is due before t_stop or max_blocks blocks are done -- no per-block call overhead on
 * the caller's side.  HOST outputs: *t_next (time of the next block that was NOT integrated, or of the last one
 * tried), the number of blocks and of particle steps taken.  An error of a step (e.g. NB_EOVERFLOW) ends the
 * loop and is returned; the counters tell how far it got. */
int nb_ac_run(nb_ctx *ctx, double eta_I, double eta_R, double dt_max, double t_stop, int64_t max_blocks,
              double *t_next, int64_t *blocks, int64_t *irregular_steps, int64_t *regular_steps);
int nb_run_blocks(nb_ctx *ctx, const double *h2_all, double eta, double dt_max, double t_stop,
                  int64_t max_blocks, double *t_next, int64_t *blocks, int64_t *particle_steps);

/* Radius control in mid-run (the paper's codes adapt the neighbour radius at regular steps; here the policy is the
 * caller's, the library only stores the radii, reading R38).  nb_ac_set_radii replaces the stored SQUARED radius of the
 * bodies idx[0..n) (DEVICE; indices outside [0, N) are ignored) by h2[0..n) (DEVICE), or of all bodies if idx == NULL
 * and n == N.  A new radius takes effect at that body's NEXT regular step, where the list is rebuilt anyway (the
 * regular force w.r.t. the old list is total - irregular(old list), so old and new radius need not agree).  Enqueued on
 * the stream.  NB_ESTATE without a live two-level state.
 * Recovery from NB_EOVERFLOW: nb_ac_step / nb_ac_run left the state untouched and the same block is due again.
 * nb_ac_get_failed tells which regular steps it attempted: *n_rows (HOST) = their number (0 if the last step did not
 * overflow), idx[0..min(n_cap, *n_rows)) (DEVICE, may be NULL) = the bodies, ascending, nnb[...] (DEVICE, may be NULL)
 * = the TRUE number of neighbours each new list would have held (those > nb_cap overflowed).  Shrink those radii
 * -- e.g. h2 *= (target / nnb)^(2/3) --, nb_ac_set_radii, and call nb_ac_step again: the block is redone with them. */
int nb_ac_set_radii(nb_ctx *ctx, int32_t n, const int32_t *idx, const double *h2);
int nb_ac_get_failed(nb_ctx *ctx, int32_t n_cap, int32_t *n_rows, int32_t *idx, int32_t *nnb);

/* Inspection: copies of the AC state into the caller's DEVICE buffers (any may be NULL): the last block's
 * idx_act[N] / idx_reg[N] (first n_irr / n_reg entries valid), aI, jI, aR, jR [N][3], tR, dtR [N], nnb[N],
 * nblist[N][nb_cap].  (x0, v0, total a0 / j0, t0 and dtI come from nb_get_state.) */
int nb_ac_get(nb_ctx *ctx, int32_t *idx_act, int32_t *idx_reg, double *aI, double *jI, double *aR, double *jR,
              double *tR, double *dtR, int32_t *nnb, int32_t *nblist);

/* Inspection / checkpoint: the stored FP64 state in the caller's layout: m[N], x0[N][3], v0[N][3],
 * a0[N][3], j0[N][3], t0[N] and (optional, may be NULL) the steps dt[N]. */
int nb_get_state(nb_ctx *ctx, double *m, double *x0, double *v0, double *a0, double *j0, double *t0,
                 double *dt);

/* ---- j-sharding ("each GPU has a similar particle dataset size ...
 * all GPUs in the same node together access the complete particle dataset").  A context then holds a
 * contiguous SHARD of the bodies -- nb_open(N_shard), nb_set_j of the shard's bodies, nb_predict_all(t)
 * -- and nb_set_j_offset gives the global index of its body 0.  nb_regular_shard sums the shard's
 * contribution to the regular force of ANY active block: idx_i[k] are GLOBAL indices and the active
 * particles' own FP64 state arrives as istate[14][n_i] (rows m, x0[3], v0[3], a0[3], j0[3], t0 -- the
 * component order of the arguments of nb_set_j), predicted to t with the predictor's own arithmetic, so
 * that a particle of this shard meets its own record at r = 0 exactly and is skipped by global index.
 * Outputs are this shard's PARTIAL results: acc, jerk, pot over the shard's j; nnb = neighbours found
 * in the shard; nblist rows = their GLOBAL indices, ascending; overflow = (nnb > nb_cap) for the shard
 * alone.  The caller adds acc / jerk / pot / nnb over the shards (an all-reduce of 7 doubles + 1 int per
 * active particle), concatenates the list rows in shard order (= ascending j) and sets
 * overflow = total nnb > nb_cap.  n_i may exceed the shard size.  DEVICE pointers.
 * Requires nb_predict_all(t) with the same t (checked: NB_ESTATE otherwise).  nb_regular / nb_regular_all on
 * a context with an offset keep LOCAL indices in and out; nb_step_host returns NB_ESTATE there. */
int nb_set_j_offset(nb_ctx *ctx, int64_t j_offset);
int nb_regular_shard(nb_ctx *ctx, double t, int32_t n_i, const int32_t *idx_i, const double *istate,
                     const double *h2_i, double *acc, double *jerk, double *pot, int32_t *nnb,
                     int32_t *nblist, int32_t *overflow);

/* ---- Block selection for callers that must not allocate (P:47 block time steps; section 3.3.1: the search
 * for the particles due next).  Same result as nb_set_steps + nb_next_block, without a context.
 *
 * Use it where a cudaMalloc is not an option: inside an application whose own memory pool has already claimed the
 * device (a stray allocation fails or eats into its budget), inside a hook that runs beside other streams and must
 * not trigger the device-wide synchronisation that cudaMalloc / cudaFree imply, or after an out-of-memory condition.
 * nb_open allocates the j-state, so none of the context calls qualify; this one makes no allocation of its own, host or
 * device: it calls neither cudaMalloc / cudaFree nor any routine that allocates.
 *
 * Inputs, DEVICE: t0[N], dt[N] (time of the last step and current step of every body).  Outputs, DEVICE, caller-owned:
 * idx_act with room for N int32 -- the bodies with t0 + dt == min_j (t0_j + dt_j), ascending, in its first n entries,
 * the rest untouched --, block[2] = {t_next, (double) n}.  Enqueued on cuda_stream (NULL = the legacy default stream)
 * on the CURRENT device; returns without synchronising, outputs valid once that stream has been synchronised.
 * Three kernels and one 8-byte memset.
 *
 * Working memory: a fixed 33,024-byte array inside the library image (the running minimum and one count per 2048
 * bodies).  Every GPU that loads libnbreg holds it from load until the process exits.  Hence the LIMIT:
 * N <= NB_STATIC_MAX_N = 16,777,216; a larger N returns NB_ELIMIT before anything is launched or written.
 * The array is shared by all calls of the process on that device and keeps the last call's contents; the call resets
 * the part that must start clean (the minimum) on the stream, in order, before its kernels.  Two calls whose GPU
 * work can OVERLAP -- different streams without an event between them, or two host threads on different streams --
 * race on it and return garbage; calls on one stream, or ordered by events, are safe.
 * The FIRST call on each device looks up the array's device address (and the SM count) and keeps it; that look-up may
 * initialise the device's CUDA context and load the library's kernels, so make one call per device during start-up,
 * before any stream capture begins.  Later calls only enqueue.
 * Errors: NB_EINVAL (NULL pointer, N <= 0), NB_ELIMIT, NB_ECUDA (the look-up or a launch failed -- e.g. the current
 * device is not sm_100; not sticky, there is no context to stick to). */
#define NB_STATIC_MAX_N 16777216
int nb_next_block_static(int64_t N, const double *t0, const double *dt, int32_t *idx_act, double *block,
                         void *cuda_stream);

/* Tuning / introspection.  Keys: */
enum {
    NB_INFO_KERNEL_LAUNCHES = 0, /* get: kernels launched by this context so far                   */
    NB_INFO_LAST_JSPLIT = 1,     /* get: number of j-range splits S used by the last nb_regular    */
    NB_INFO_LAST_IBLOCK = 2,     /* get: i-particles per CTA used by the last nb_regular           */
    NB_INFO_LAST_GRID = 3,       /* get: CTAs of the last force-kernel launch                      */
    NB_INFO_SM_COUNT = 4,        /* get: multiProcessorCount of the device                         */
    NB_INFO_N_PADDED = 5,        /* get: N rounded up to the j-tile size                           */
    NB_TUNE_FORCE_JSPLIT = 16,   /* set: force S (0 = automatic)                                   */
    NB_TUNE_FORCE_VARIANT = 17,  /* set: force the kernel variant 0..4 (-1 = automatic)            */
    NB_INFO_LAST_VARIANT = 18,   /* get: kernel variant used by the last nb_regular                */
    NB_TUNE_PROFILE = 19,        /* set 1: bracket every force-kernel launch with CUDA events on the
                                    context's stream (ring of 256 launches); set 0: off, ring cleared */
    NB_INFO_FORCE_KERNEL_NS = 20,    /* get: summed device time of the bracketed force-kernel launches,
                                        in ns (synchronises the stream)                             */
    NB_INFO_FORCE_KERNEL_COUNT = 21, /* get: number of bracketed launches in that sum               */
    NB_TUNE_STEP_CHUNKS = 22,        /* set: number of chunks nb_step_host sends the j-state in, 1..8
                                        (1 = no overlap; sizes 1/2^(n-1), 1/2^(n-1), then doubling);
                                        0 = automatic (5 chunks from 524288 bodies, 3 from 131072)  */
    NB_TUNE_FUSE_PREDICT = 23,       /* set 1 (default): nb_predict_all defers its kernel; a block of <= 128
                                        active particles that follows predicts inside the force kernel
                                        (reads the FP64 state, no predicted records written), any other
                                        consumer writes the records first.  set 0: nb_predict_all launches
                                        the predictor at once and nb_regular always reads the records      */
    NB_TUNE_LOCAL_G_MILLI = 24,      /* set: 1000 G of the local-frame guard |x_i - c| <= G h_i under which a
                                        warp differences positions in its own frame (default 8000; 0 = never:
                                        hi/lo differencing everywhere)                                      */
    NB_TUNE_STATS = 25,              /* set 1: count, from now on, the warps of the force kernel and those
                                        that took the local frame; set 0: off                               */
    NB_INFO_LOCAL_WARPS = 26,        /* get: warps that took the local frame since NB_TUNE_STATS was set    */
    NB_INFO_TOTAL_WARPS = 27,        /* get: all warps since then (both synchronise the stream)             */
    NB_INFO_LAST_FUSED = 28,         /* get: 1 if the last nb_regular predicted inside the force kernel     */
    NB_TUNE_REORDER_MIN = 29,        /* set: blocks of at least this many active particles are put in Morton
                                        order inside the library before the force kernel, so that the 64
                                        particles of a warp sit close together and take the local frame
                                        (default 4096; 0 = never).  Outputs keep the caller's order.        */
    NB_INFO_LAST_REORDERED = 30,     /* get: 1 if the last block was reordered                              */
    NB_TUNE_SPECULATE = 31,          /* set 1 (default): nb_block_step enqueues the chain of a SMALL block (size class
                                        of the previous one: 32 / 64 / 128) before the host has read {t_next, n}: the
                                        kernels take both from device memory and do nothing if the block is larger,
                                        in which case the ordinary launches follow.  set 0: always wait for n      */
    NB_INFO_SPEC_HITS = 32,          /* get: blocks integrated by a speculative chain                               */
    NB_INFO_SPEC_MISSES = 33,        /* get: speculative chains that turned out to be no-ops                        */
    NB_TUNE_SELECT_CHUNKS = 34,      /* set 1 (default): the block loops keep min (t0 + dt) per chunk of 2048 bodies between
                                        blocks and rescan only the chunks the last corrector touched (the search for
                                        the due particles must not cost O(N) per block); 0 = scan all N every block.  The
                                        selected blocks do not depend on it                                            */
    NB_TUNE_IRR_PRED_MIN = 35,       /* set: the neighbour force of a block of at least this many bodies (default 49152; 0 =
                                        never) predicts every body once into 64 B records and gathers those instead of
                                        predicting each listed neighbour from its 128 B state line.  Same bits either way   */
    NB_INFO_LAST_BLOCK_N = 36,       /* get: bodies in the last block integrated by nb_block_step / nb_run_blocks (0: none,
                                        or the last loop was the two-level one)                                         */
    NB_TUNE_SELECT_GRID = 37,        /* set: upper limit on the CTAs of the block loops' scatter kernel (0 = none, default).  The
                                        library already limits that grid to what the device holds at once, because a CTA waits
                                        for the counts of the chunks before its own; each CTA then takes several chunks of 2048
                                        bodies in ascending order.  A smaller limit exercises that route at small N (tests);
                                        the selected blocks do not depend on it                                           */
    NB_INFO_FORCE_KERNEL_NS_AT = 1000 /* get, key = 1000 + q (q < 256): device time in ns of the q-th bracketed
                                        force-kernel launch since NB_TUNE_PROFILE was set (synchronises)    */
};
int nb_get_info(nb_ctx *ctx, int32_t key, int64_t *value);
int nb_set_tuning(nb_ctx *ctx, int32_t key, int64_t value);

/* Launch planning as pure host functions (no device, no context): what nb_regular would launch for a
 * block of n_i out of N bodies on a device with sm_count SMs holding ctas_per_sm force-kernel CTAs
 * each -- kernel variant (0: 512, 1: 256, 2: 128, 3: 64, 4: 32 i-particles per CTA), its i-block, the number
 * of j-range splits and the j-tiles (256 bodies) per split; and the chunks nb_step_host sends the
 * j-state in (chunks = 0: automatic): first_body[0..*nchunk] (room for 9) are the chunk boundaries. */
int nb_plan_regular(int64_t N, int64_t n_i, int32_t sm_count, int32_t ctas_per_sm, int32_t *variant,
                    int32_t *iblock, int32_t *jsplit, int32_t *tiles_per_split);
int nb_plan_chunks(int64_t N, int32_t chunks, int64_t *first_body, int32_t *nchunk);

int nb_last_cuda_error(nb_ctx *ctx); /* cudaError_t of the sticky failure, 0 if none */
const char *nb_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* NBREG_H */
