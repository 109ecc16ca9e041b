/* sledge.h -- C ABI of the B200-native sledgehamr hot path (arXiv 2404.02950).
 *
 * One library, libsledge.so, hand-written CUDA for sm_100a.  No torch types, no exceptions, no CPU
 * fallback: every compute entry point launches kernels on the CUDA stream given at create time and
 * returns immediately (asynchronous), or fails with a negative code.
 *
 * Citations are PAPER.md line numbers (text of arXiv 2404.02950) and DESIGN.md readings (R#).
 *
 * Grid (Eq.1-3): level l has the periodic index space [0, n0*2^l)^3, spacing
 * h_l = h0/2^l, and is covered by rectangular boxes whose low corner and size are multiples of
 * blocking_factor; level 0 covers the domain; level l+1 is properly nested in level l (L70, L137).
 * State per cell: u = (psi1, psi2, Pi1, Pi2) (L189-190), component index 0..3 in that order.
 *
 * Device layout: per level, 4 state buffers; a buffer is two
 * planes, PSI = interleaved (psi1,psi2) pairs and PI = interleaved (Pi1,Pi2) pairs, boxes stored back
 * to back, each box with nghost ghost layers and its x rows padded to 128-byte multiples.
 *
 * Ownership: the caller allocates ONE device arena (sledge_arena_bytes tells how large) and lends
 * it for the lifetime of the context; the library never allocates device memory.  All `dev_`
 * pointers are device pointers, all `host_` pointers are host pointers (pinned for async copies).
 *
 * Errors: 0 on success, a negative sledge_status otherwise; sledge_last_error() returns the text.
 */
#ifndef SLEDGE_H
#define SLEDGE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sledge_ctx sledge_ctx; /* opaque; host-side metadata only */

typedef enum {
  SLEDGE_OK = 0,
  SLEDGE_EINVAL = -1, /* bad parameter / overlapping, misaligned or non-nested boxes            */
  SLEDGE_ENOMEM = -2, /* arena too small or misaligned                                           */
  SLEDGE_ECUDA = -3,  /* CUDA runtime / launch error (no device, bad stream, kernel fault)       */
  SLEDGE_ESTATE = -4  /* call not valid in the current state (e.g. rk_stage out of order)        */
} sledge_status;

enum { SLEDGE_F32 = 0, SLEDGE_F64 = 1 };
enum { SLEDGE_RK_LEAN = 0, SLEDGE_RK_CLASSIC = 1, SLEDGE_RK_FUSED = 2, SLEDGE_RK_FUSED3 = 3 };

/* Inclusive cell range lo..hi of one box in the index space of `level`; axis order x, y, z. */
enum { SLEDGE_INTERP_TRILINEAR = 0, SLEDGE_INTERP_QUARTIC = 4 };
enum { SLEDGE_NCOMP = 4, SLEDGE_NCOMP_GW = 16, SLEDGE_RKN_MAX_STAGES = 5 };

typedef struct {
  int32_t level;
  int32_t lo[3];
  int32_t hi[3];
} sledge_box;

typedef struct {
  int32_t n_levels;        /* 1..8                                                                */
  int32_t n0[3];           /* level-0 cells per axis, periodic (L23); multiples of blocking_factor */
  int32_t nghost;          /* ghost layers per box (L68-70, L772): lap_order <= nghost < blocking_factor */
  int32_t blocking_factor; /* power of 2 (L39, L771)                                              */
  int32_t dtype;           /* SLEDGE_F32 / SLEDGE_F64: storage AND arithmetic type                */
  int32_t lap_order;       /* paper's `order` (L649): 1 = 7-, 2 = 13-, 3 = 19-point Laplacian      */
  int32_t eta_fixed;       /* 1 = Minkowski test variant: eta_s = eta for every stage (R3)         */
  int32_t rk_dataflow;     /* words moved per cell-step (R5): SLEDGE_RK_FUSED 20 (two stages per sweep, on every
                              level; a level falls back to LEAN only with quartic interpolation and nghost = 1),
                              SLEDGE_RK_LEAN 52, SLEDGE_RK_CLASSIC 64; sledge_level_dataflow tells what runs.
                              In fp64 SLEDGE_RK_FUSED runs the "W form": the second sweep
                              recovers Pi of the third stage as (W - 2 psi) / dt, an absolute error of about
                              2^-53 * 2 |psi| / dt per step (1e-14 for dt = 0.025): SLEDGE_RK_FUSED3 is the same
                              two-sweep flow without that term (three differenced fields in the second sweep,
                              ~7 % slower), for very small dt; fp32 always runs it                            */
  double h0;               /* level-0 spacing, Eq.1                                               */
  double lambda;           /* Eq.11 generalised (R2): k_Pi = -(friction/eta) Pi + Lap psi          */
  double a_mass;           /*        - lambda eta^2 psi (psi1^2+psi2^2-1) - a_mass psi             */
  double friction;         /* paper: 2 (Eq.11); BASELINE.json configs: 0                          */
  double ko_strength[4];   /* Kreiss-Oliger dissipation (Eq.7): epsilon_KO >= 0 of psi1, psi2, Pi1, Pi2
                              (sim.dissipation_strength[_$ScalarField], L749-750); all 0 = term removed.
                              Q_l u = (-1)^(r+1) eps h_l^(2r-1) / 2^(2r) * sum_d d^(2r)u/dx_d^(2r) is added to the
                              RHS of every component, the derivative as the (2r+1)-point central difference.
                              With the term on, every level runs the staged LEAN / CLASSIC sweeps (FUSED needs
                              k_psi = Pi pointwise) and the stage fills move Pi ghosts as well.          */
  int32_t ko_order;        /* r = sim.dissipation_order in {2,3} = ghost cells the term needs (L751): r <= nghost */
  int32_t integrator;      /* integrator.type (L808): 0 or 4 = classic RK4; 3 or 10 = SSPRK3 (Shu-Osher form,
                              three state buffers, 32 words per cell-step; rk_dataflow is ignored); 20 = the user's
                              Runge-Kutta-Nystrom tableau below (rk_dataflow is ignored)                  */
  int32_t interp;          /* coarse->fine ghost interpolation (L70-72): SLEDGE_INTERP_TRILINEAR = cell-centred
                              trilinear, weights 3/4, 1/4 per axis (BASELINE.json config 5); SLEDGE_INTERP_QUARTIC =
                              amr.interpolation_type 4, the paper's default (L780): per axis the quartic matching the
                              averages of the coarse cells c0-2..c0+2, averaged over the fine cell,
                              c0 -+ (3 c[-2] - 22 c[-1] + 22 c[+1] - 3 c[+2])/128, tensor product; both linear in time.
                              Quartic needs ceil(nghost/2) + 2 <= blocking_factor/2 on a multi-level hierarchy. */
  int32_t shadow_level;    /* 1 = reserve room in the arena for the shadow level of level 0 (L98): a coarsened copy of
                              level 0 (spacing 2 h0, one periodic box) that sledge_shadow_tee evolves; n0 must be even */
  int32_t gw;              /* sim.gravitational_waves (L404): 1 = every cell also carries the auxiliary fields of Eq.16,
                              components 4..9 = Gw::u_xx, u_yy, u_zz, u_xy, u_xz, u_yz and 10..15 = Gw::du_xx .. du_yz
                              (L436), evolved with (R25, conformal-time form of Eq.16 like Eq.9-11)
                                k_u_ij = du_ij,  k_du_ij = -(gw_friction/eta) du_ij + Lap u_ij + gw_coupling T_ij,
                                T_ij = sum_c d_i psi_c d_j psi_c,  Laplacian<lap_order> and Gradient<lap_order> (L649-658).
                              Classic RK4 only; the scalar sector then runs the staged LEAN / CLASSIC sweeps (the
                              source needs psi of every stage state), the auxiliary fields the LEAN data-flow;
                              trilinear coarse->fine interpolation only.                                        */
  int32_t rkn_stages;      /* integrator 20: stages s of the tableau, 1..5                                     */
  double gw_coupling;      /* Eq.16's 16 pi G in the project's units                                           */
  double gw_friction;      /* Eq.16's 3H written like Eq.11's 2/eta: friction term (gw_friction / eta) du_ij    */
  /* integrator.type 20 (L808-815 Table V; R26): explicit Runge-Kutta-Nystrom scheme for
   * psi'' = f(psi, eta) = Lap psi - psi (lambda eta^2 (|psi|^2 - 1) + a_mass); friction and ko_strength must be 0:
   *   Psi_i = psi + c_i dt Pi + dt^2 sum_{j<i} a_ij f_j,  f_i = f(Psi_i, eta + c_i dt)
   *   psi' = psi + dt Pi + dt^2 sum_i barb_i f_i,          Pi' = Pi + dt sum_i b_i f_i                        */
  double rkn_nodes[6];         /* rkn.nodes c (L814); entries past rkn_stages are ignored                      */
  double rkn_weights_b[6];     /* rkn.weights_b (L812)                                                          */
  double rkn_weights_bar_b[6]; /* rkn.weights_bar_b (L813)                                                      */
  double rkn_tableau[21];      /* rkn.tableau (L815): flattened lower triangle INCLUDING the diagonal, row i =
                                  a_i0 .. a_ii; the diagonal must be 0 (explicit schemes only)                  */
} sledge_params;

/* Size of the device arena needed for this hierarchy.  Host-only: validates params and boxes
 * (same checks as sledge_create) and needs no GPU.  ctx-less errors: sledge_last_error(NULL). */
int sledge_arena_bytes(const sledge_params* params, const sledge_box* boxes, int nbox, size_t* bytes);

/* Build a context.  dev_arena: device memory, 256-byte aligned, >= sledge_arena_bytes, zero-filled
 * by this call.  cuda_stream: a cudaStream_t (0 = legacy default stream); every later call enqueues
 * on it.  Box indices used below are positions in `boxes`. */
int sledge_create(sledge_ctx** ctx, const sledge_params* params, const sledge_box* boxes, int nbox,
                  void* dev_arena, size_t arena_bytes, void* cuda_stream);
int sledge_destroy(sledge_ctx* ctx);

/* Copy one component (0..3, or 0..15 with gw) of one box between a dense device array of its valid region (x fastest,
 * nx*ny*nz reals of the context's dtype) and the current state.  Setting a state invalidates the
 * level's (old,new) pair used for temporal ghost interpolation. */
int sledge_set_state(sledge_ctx* ctx, int box, int comp, const void* dev_src);
int sledge_get_state(sledge_ctx* ctx, int box, int comp, void* dev_dst);
/* Same with HOST buffers (pinned memory for truly asynchronous copies).  The library stages through slots inside
 * the arena (two for uploads, four for downloads) and runs the host<->device copies on two streams of its own, ordered against the
 * context stream with events: the upload of component c+1 overlaps the repacking kernel of c, downloads drain while
 * the context stream goes on, and the downloads of one step overlap the uploads of the next (PCIe is full duplex).
 * Ordering seen by the caller is that of the context stream: a set is complete for every later call on the context;
 * a get has delivered its data after sledge_synchronize, or once work enqueued after sledge_host_copies_join runs. */
int sledge_set_state_host(sledge_ctx* ctx, int box, int comp, const void* host_src);
int sledge_get_state_host(sledge_ctx* ctx, int box, int comp, void* host_dst);
/* Make the context stream wait for every host copy enqueued so far (e.g. before recording an event that should
 * include the downloads). */
int sledge_host_copies_join(sledge_ctx* ctx);
/* One component of one box INCLUDING ghosts: (nx+2g)*(ny+2g)*(nz+2g) reals, x fastest.  Ghost values are those of
 * the last fill that touched them: sledge_fill_ghosts fills every ghost cell of all four components; the fills
 * inside a step move psi only unless Pi is differenced (FUSED sweeps, Kreiss-Oliger term), R10; before a FUSED sweep
 * of a level > 0 the Pi ghost cells that are interpolated from the coarse level do NOT hold Pi but the finite
 * difference in time of the interpolated coarse psi between the sweep's two stage times (what the sweep needs to form
 * the later stage's psi there, L72), so after a step only sledge_fill_ghosts makes the ghost contents meaningful. */
int sledge_get_ghosted(sledge_ctx* ctx, int box, int comp, void* dev_dst);

/* Ghost fill of the CURRENT state of `level` (L68-74): every psi ghost cell <- the valid cell of the
 * same level at the periodically wrapped index if one exists, else trilinear interpolation of the
 * next coarser level, itself linearly interpolated in time between its states at the start and end
 * of its last step (alpha = (time - t_old)/(t_new - t_old); the current coarse state alone if that
 * level has not stepped since its state was set).  This explicit call fills EVERY ghost cell (psi and Pi).
 * The fills that sledge_rk_step / sledge_rk_stage issue themselves move only the ghost cells the Laplacian's star
 * stencil reaches (outside the box along one axis, by at most lap_order), and none at all on a level that is one
 * box over the periodic domain (the kernels read the wrapped cell directly); with quartic interpolation and
 * nghost >= 2 a fill of level l > 0 first refreshes, where stale, the whole ghost shell of level l-1's old and new
 * states with same-level copies (the 5^3 windows are read through them).  So after a step the ghost contents
 * are unspecified until this function is called. */
int sledge_fill_ghosts(sledge_ctx* ctx, int level, double time);

/* One classic-RK4 stage (integrator.type 4, L808) of `level`: ghost fill of the stage input at
 * eta + c_s dt, then the fused Laplacian + potential + stage-update kernel (Eq.10-11).  stage =
 * 0,1,2,3 in order; `eta` is the time at the START of the step for all four calls.  Stage 3 makes
 * the new state current.  With integrator 3 / 10 (SSPRK3) stages 0,1,2 are the scheme's three stages
 * (c = 0, 1, 1/2), stage 2 makes the new state current and stage 3 is a no-op.
 * Test / timing hook; sledge_rk_step is built from it. */
int sledge_rk_stage(sledge_ctx* ctx, int level, int stage, double dt, double eta);

/* ONE coarse step eta -> eta + dt of the whole hierarchy (L64-76, L88 Fig.2): level l takes 2^l steps
 * of dt/2^l (Eq.3) with per-stage ghost fills, finest first to finish, average-down after each pair
 * of fine steps.  Afterwards the valid cells of every level hold the state at eta + dt; ghost
 * contents are unspecified until the next sledge_fill_ghosts. */
int sledge_rk_step(sledge_ctx* ctx, double dt, double eta);

/* String tagging (L349-371 hook; rule: DESIGN.md R8) of the current state of `level`, ghosts filled
 * first.  dev_tags: one byte per valid cell, boxes of the level back to back in box order, x fastest;
 * bit0/1/2 = the xy / yz / zx plaquette whose lowest corner is the cell has non-zero winding.
 * dev_counts: uint32 per aligned 32^3 block of the level's index space (x fastest,
 * ceil(n/32) per axis) = number of tagged cells in it; zeroed by the call.  Either may be NULL. */
int sledge_tag_strings(sledge_ctx* ctx, int level, uint8_t* dev_tags, uint32_t* dev_counts);

/* String tagging with NO allocation anywhere: no context, no arena.  For callers that cannot call cudaMalloc (code
 * under CUDA graph capture, tight serving loops, harnesses that forbid it).  Tags ONE periodic box given as two dense
 * device arrays -- the same rule, kernel (k_tag_strings) and output layout as sledge_tag_strings on a one-box level 0.
 *   dev_psi1, dev_psi2 : device, nx*ny*nz reals each of `dtype` (SLEDGE_F32 / SLEDGE_F64), x fastest; read only.
 *   n                  : HOST, {nx, ny, nz}, each >= 2; the box is periodic in all three directions (L23).
 *   dev_tags           : device, one byte per cell, x fastest (bit0/1/2 as above); may be NULL.
 *   dev_counts         : device, uint32 per aligned 32^3 block (x fastest, ceil(n/32) per axis); zeroed by the call;
 *                        may be NULL.
 *   cuda_stream        : a cudaStream_t (0 = legacy default stream); the call enqueues on it and returns.
 * Scratch: the kernel reads pair-interleaved, 128-byte-aligned rows, so the call first packs
 * the two arrays into that layout -- together with its box / tile tables -- inside a file-scope
 * `static __device__` array of SLEDGE_STATIC_SCRATCH_BYTES (8 MiB; every GPU that loads the library holds it until the
 * process exits).  A box whose packed size exceeds it is rejected with SLEDGE_EINVAL and a text that names the limit
 * (fits: 72^3 in fp64, 88^3 in fp32; bytes = 256 + 20 per tile, rounded up to 256, + 2 * sizeof(real) * pitch *
 * (ny + 2) * (nz + 2) with pitch = nx + 9 (fp64) / nx + 17 (fp32) cells rounded up to 128 bytes).  The call runs on the device that owns dev_psi1 and
 * calls no cudaMalloc, cudaFree or allocating library routine, and copies nothing from host memory.
 * Every call shares the one array per device, which keeps the previous call's contents (everything a call reads it
 * has written itself first): calls whose kernels may overlap on the GPU (different streams, no ordering between
 * them) RACE -- order them on one stream or with events.  Errors: SLEDGE_EINVAL (null / non-device pointer, bad n,
 * dtype, too large), SLEDGE_ECUDA; text by sledge_last_error(NULL). */
#define SLEDGE_STATIC_SCRATCH_BYTES (8u << 20)
int sledge_tag_strings_static(const void* dev_psi1, const void* dev_psi2, const int* n, int dtype, uint8_t* dev_tags,
                              uint32_t* dev_counts, void* cuda_stream);

/* Level synchronisation (L74): every cell of level fine_level-1 covered by fine_level <- mean of its 8
 * children, all four components, on the current states. */
int sledge_average_down(sledge_ctx* ctx, int fine_level);

/* Truncation-error (TEE) tags of the self-shadow method (L82-111 Eq.5-6, L373-380 Eq.12 with f = identity), fused
 * into the synchronisation: from now on every average-down of `fine_level` -- the explicit call above and the ones
 * inside sledge_rk_step -- first compares, for every coarse cell C under a fine box, the coarse level's own value
 * with the mean of its 8 fine children, Delta_c = |phi_c^{l-1}(C) - mean_c| for every component c = psi1, psi2, Pi1,
 * Pi2 (in the context's dtype), and gives the 8 children the tag byte  sum_c (Delta_c > eps4[c]) << c  (strict >,
 * Eq.12); then it overwrites the coarse value as before.
 *   eps4       : HOST, four thresholds >= 0 (amr.te_crit_$ScalarField, L781-782; the momenta are members of the
 *                Scalar set, L202); DBL_MAX or +inf -- the paper's default -- leaves a component untagged.
 *   dev_tags   : device, one byte per VALID cell of `fine_level`, boxes of the level back to back in input order,
 *                x fastest (the layout of sledge_tag_strings); 2-byte aligned; may be NULL.
 *   dev_counts : device, uint32 per aligned 32^3 block of the fine level's index space (x fastest), zeroed and
 *                refilled at every synchronisation: tagged fine cells in the block; may be NULL.
 * Both NULL switches the tags off.  The buffers stay owned by the caller and must stay valid while enabled.  A level
 * synchronises once per step of its parent, so after sledge_rk_step the buffers hold the LAST synchronisation.
 * Level 0 has no coarser partner: SLEDGE_EINVAL here; its tags come from sledge_shadow_tee below. */
int sledge_tee_enable(sledge_ctx* ctx, int fine_level, const double* eps4, uint8_t* dev_tags,
                      uint32_t* dev_counts);

/* Truncation-error tags of LEVEL 0 through the shadow level (L98: "we do indeed introduce such a coarsened version of the
 * coarse level ... only evolved for a single time step Delta t_s = 2 Delta t_{l=0}"; R27).  Needs
 * shadow_level = 1 at create.  The call (1) fills the shadow level with the mean of the 8 level-0 children of each of
 * its cells (K4 run into the shadow box), (2) advances the shadow level by ONE step of 2 dt from eta (same equation,
 * spacing 2 h0, periodic) and the hierarchy by TWO coarse steps of dt (as two sledge_rk_step calls at eta and eta + dt),
 * (3) compares, for every shadow cell C, Delta_c = |shadow_c(C) - mean of its 8 level-0 children| with eps4[c] and gives
 * the 8 children the tag byte sum_c (Delta_c > eps4[c]) << c (the K4 TEE kernel of sledge_tee_enable, coarse side =
 * the shadow box).  dev_tags: one byte per valid level-0 cell, boxes back to back in input order, x fastest, 2-byte
 * aligned; dev_counts: uint32 per aligned 32^3 block of level 0, zeroed by the call; either may be NULL.  Afterwards the
 * hierarchy is at eta + 2 dt and the shadow level's contents are dead (it is rebuilt by the next call). */
int sledge_shadow_tee(sledge_ctx* ctx, double dt, double eta, const double* eps4, uint8_t* dev_tags, uint32_t* dev_counts);

/* Bookkeeping. */
int sledge_level_cells(const sledge_ctx* ctx, int level, int64_t* valid_cells, int64_t* count_blocks);
int64_t sledge_launch_count(const sledge_ctx* ctx); /* kernels launched by this context so far */
/* Storage layout of `level` ("storage boxes"): the boxes given to sledge_create are coalesced
 * into larger rectangles wherever two of them share a whole face, so that no ghost cells lie between them; every entry
 * point still addresses the caller's boxes (box index, tag layout, dense copies).  storage_boxes: rectangles the level
 * is stored in (= the caller's box count of that level when nothing could be merged, or with SLEDGE_COALESCE=0 in the
 * environment at create); stored_cells: cells per plane of one state buffer, ghost layers and row padding included.
 * Either pointer may be NULL.  SLEDGE_EINVAL for a bad level. */
int sledge_level_storage(const sledge_ctx* ctx, int level, int* storage_boxes, int64_t* stored_cells);
/* The data-flow `level` runs: K1 launches per step of that level (the auxiliary-field stages of
 * gw included) and algorithmic words (reals read + written) per cell-step of those launches: FUSED 2 / 20 (level 0, and
 * finer levels unless quartic interpolation runs per cell, nghost = 1), LEAN 4 / 52, CLASSIC 4 / 64, SSPRK3 3 / 32, RKN s / sum over the
 * stages, plus 4 / 164 with gw.  bench.py's roofline numerator. */
int sledge_level_dataflow(const sledge_ctx* ctx, int level, int* k1_launches_per_step, int* words_per_cell_step);

/* Wait for everything enqueued so far and report deferred errors: SLEDGE_ECUDA for a kernel fault,
 * SLEDGE_ESTATE if a kernel met a ghost or coarse cell that no box provides (cannot happen for box
 * lists that passed sledge_create's nesting check).  The only blocking call besides
 * sledge_profile_read and sledge_destroy. */
int sledge_synchronize(sledge_ctx* ctx);

/* Per-kernel device timing with CUDA events on the context stream (bench.py's roofline leg).
 * kind: 0 = rk stage kernel, 1 = ghost fill, 2 = tagging, 3 = average-down.  While enabled every
 * launch of that kind is bracketed by an event pair (at most 4096 pairs are kept).
 * sledge_profile_read synchronises the stream and returns launches and their summed milliseconds
 * since the last enable. */
int sledge_profile_enable(sledge_ctx* ctx, int on);
int sledge_profile_read(sledge_ctx* ctx, int kind, int64_t* launches, double* total_ms);

/* Text of the last error of this context (or of the last failed ctx-less call if ctx == NULL). */
const char* sledge_last_error(const sledge_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* SLEDGE_H */
