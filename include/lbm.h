/* lbm.h — C ABI of the B200-native fused D3Q19 LES + forest-canopy lattice Boltzmann step.
 *
 * Method: arxiv 2206.15454 (Shao et al.), Algorithm 1 with Eqs. 1-16:
 *   stream (Eq. 1) -> moments (Eqs. 5-7) -> forest drag F_f = -C_D a_f(y)|u|u
 *   (Eq. 13) with the half-force velocity shift (Eq. 6) -> Smagorinsky relaxation
 *   time from the local non-equilibrium momentum flux (Eqs. 10-12) -> BGK collision
 *   (Eqs. 2-3) with Guo forcing (Eq. 4); periodic x/z and no-slip wall without a
 *   wall function (L177, L216); time + x-z-plane averages of velocity and stresses (L200, L251).
 *   The readings of ambiguous passages are listed in DESIGN.md ("Readings", R1..R26).
 *
 * Conventions
 *   - Lattice units: dx = dt = 1, c_s^2 = 1/3.  x streamwise, y wall-normal, z spanwise.
 *   - cell = x + nx*(y + ny*z) (x fastest).  All ny rows are fluid; the bottom boundary plane is
 *     the face below row 0 and the top boundary plane the face above row ny-1 (halfway links).
 *   - x and z are always periodic.
 *   - Every call returns LBM_OK (0) or a negative lbm_status; no exception or abort crosses the
 *     ABI.  lbm_last_error() returns a thread-local, NUL-terminated description of the last
 *     failure on the calling thread.
 *   - "dev" pointers are CUDA device pointers, "host" pointers are ordinary host pointers.  The
 *     library never allocates population memory: the caller (the Python binding uses
 *     torch.empty) owns one device workspace of lbm_workspace_bytes() bytes, 256-byte aligned,
 *     and must keep it alive until lbm_destroy.  All kernels are launched on the CUDA stream
 *     given to lbm_bind (a cudaStream_t passed as void*; NULL = legacy default stream), which
 *     must belong to the device that holds the workspace.  lbm_bind records that device and every
 *     later call runs under it (the caller's current device is restored on return).
 *   - All calls on one handle must come from one host thread at a time.
 *   - Time: "state k" is the post-collision population set after k steps.  The sample
 *     S_k = (rho, u) is obtained by streaming state k and applying Eqs. 5-6 and 13 (what step
 *     k+1 sees before colliding; reading R19).  lbm_step(1) maps state k -> k+1 and, when
 *     statistics are on and due, accumulates S_k.  lbm_get_macros returns S_k, state unchanged.
 */
#ifndef LBM_B200_H
#define LBM_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lbm_s lbm_t; /* opaque, owned by the library */

typedef enum lbm_status {
    LBM_OK = 0,
    LBM_EINVAL = -1,    /* bad argument (size, nu <= 0, NULL pointer, unsupported flag combination) */
    LBM_ENOMEM = -2,    /* workspace too small / misaligned, or host allocation failed */
    LBM_ESTATE = -3,    /* call out of order (step before bind/init, ...) */
    LBM_ECUDA = -4,     /* CUDA runtime error; text in lbm_last_error() */
    LBM_EDIVERGED = -5  /* a non-finite density was seen by the statistics / macros reduction */
} lbm_status;

/* bc_flags bit field */
#define LBM_BOTTOM_WALL       0u          /* bits 0-1: halfway bounce-back no-slip wall (L177, L216) */
#define LBM_BOTTOM_PERIODIC   1u          /*           periodic in y (closed-form test cases only)   */
#define LBM_TOP_WALL          (0u << 2)   /* bits 2-3: halfway bounce-back                            */
#define LBM_TOP_FREE_SLIP     (1u << 2)   /*           specular reflection (BASELINE.json configs)    */
#define LBM_TOP_PERIODIC      (2u << 2)   /*           periodic in y (must pair with BOTTOM_PERIODIC) */
#define LBM_TOP_FORCED_EQ     (3u << 2)   /*           forced-equilibrium lid, the paper's ABL top (L216) */
#define LBM_DRAG_VECTOR       (1u << 4)   /* bit 4: 0 streamwise-only drag (paper, L98/L103), 1 vector */
#define LBM_SOLID_MASK        (1u << 5)   /* bit 5: per-cell geometry: solid bit mask (lbm_set_solid) and
                                             forest codes (lbm_set_forest_codes)                            */
#define LBM_STORAGE_AA        (1u << 6)   /* bit 6: 0 two-lattice pull, 1 single-array AA pattern     */
#define LBM_Z_HALO            (1u << 7)   /* bit 7: z slab of a larger lattice: planes 0 and nz-1 are ghost
                                             planes served by the halo calls, planes 1..nz-2 are updated
                                             (any storage scheme)                                           */
#define LBM_VEC_SHIFT         8           /* bits 8-10: cells per thread override (0 auto, 1, 2, 4)   */
#define LBM_VEC_MASK          (7u << 8)
#define LBM_STORAGE_AAX       (1u << 11)  /* bit 11: single array, x-balanced AA pattern: as LBM_STORAGE_AA in
                                             memory and results, but both steps of the pattern carry half of
                                             the x streaming (lbm_kernels.cuh "AAX"); geometry handles too     */

#define LBM_NSTAT 10 /* columns of lbm_stats_read */

/* Initial-profile kinds for lbm_set_init */
#define LBM_INIT_POWER_LAW 0 /* U_ref * ((j+1/2)/ny)^(1/7) e_x */
#define LBM_INIT_PARABOLA  1 /* U_ref * 4 eta (1-eta) e_x, eta = (j+1/2)/ny */
#define LBM_INIT_REST      2 /* u = 0 */

/* Bytes of device workspace a handle with these sizes/flags needs (populations: 76 B/cell for
 * AA, 152 B/cell for two-lattice; plus statistics partials, tables and a host-transfer staging
 * area).  Host call, no CUDA work. */
int lbm_workspace_bytes(int nx, int ny, int nz, uint32_t bc_flags, size_t *bytes);

/* Create a handle.  Problem statement of Alg. 1's inputs (L140) and Table I/II parameters:
 *   nu          kinematic viscosity, lattice units, > 0; tau0 = 3 nu + 1/2 (R3)
 *   Cs          Smagorinsky constant; the paper's C_smag (Eq. 9) equals Cs^2 (R9)
 *   body_force  host, 3 doubles, force DENSITY F_b (Eq. 16; R4); copied; NULL = 0
 *   Cd          drag coefficient C_D of Eq. 13
 *   lad_profile host, ny doubles a_f(y_j) at cell centres y_j = j + 1/2 (Eqs. 14-15 evaluated by
 *               the caller, or lbm_lad_profile below); copied; NULL or all-zero = no forest
 * Host call; needs a CUDA device only at lbm_bind.  Errors: LBM_EINVAL, LBM_ENOMEM. */
int lbm_create(lbm_t **out, int nx, int ny, int nz, double nu, double Cs,
               const double *body_force, double Cd, const double *lad_profile,
               uint32_t bc_flags);

/* Velocity of the forced-equilibrium top (LBM_TOP_FORCED_EQ; "the top boundary is
 * forced to be in equilibrium with the same velocity as the free-stream flow"): every population
 * entering through the top face is f_eq,i(rho = 1, U_top) (Eq. 3).  U_top: host, 3 doubles,
 * copied; default 0.  May be called at any time; takes effect from the next step.
 * LBM_EINVAL if the handle was not created with LBM_TOP_FORCED_EQ or a component is not finite. */
int lbm_set_top_velocity(lbm_t *h, const double *U_top);

/* Per-cell geometry (handles created with LBM_SOLID_MASK; "a bit mask" codes the
 * cell kind, L226 turbulence-trip boxes).
 *
 * lbm_set_solid: solid_host is host, [nz][ny][nx] bytes, non-zero = solid; NULL = no solid cell.
 * The library packs it to 1 bit per cell (one 32-bit word per 32 x cells, rows padded to whole
 * words, 0.125 B/cell) in the workspace.  A link between a fluid and a solid cell is a halfway
 * bounce-back link; solid cells keep the rest state, report rho = 1, u = 0 and are left out of the
 * plane sums (the divisor of the averages stays nx*nz).  Call after lbm_bind, before or AFTER the
 * state exists: on a running handle the flow is kept (L226: "the boxes are removed from the
 * computational domain.  The flow remains in the turbulent status afterwards") - every cell that
 * stays fluid keeps its populations bit for bit, a cell that turns fluid starts at rest
 * (f = f_eq(1, 0), reading R28), a cell that turns solid is cleared; lbm_time is unchanged.
 * Synchronises the stream.  On a z slab (LBM_Z_HALO) the mask covers the two ghost planes as well
 * and every rank changes its mask at the same time step; after a change on a running handle the
 * caller repeats the halo exchange (lbm_halo_pack, exchange, lbm_halo_unpack on both faces) before
 * the next step: in the single-array storages at even time steps the populations that move
 * between a changed cell and a neighbour across a slab face are converted in the ghost planes of
 * the rank that holds them and travel with that exchange (at odd steps and in two-lattice storage
 * the exchange repeats what the planes already hold).
 *
 * lbm_set_forest_codes: heterogeneous canopies (L129-135: "The code for each forest cell contains
 * ... h ... y ... y_m ... stored into the forest cell's code using a bit mask"; Alg. 1 "if
 * forest cell").  code_host is host, [nz][ny][nx] uint32, 0 = not a coded cell (the cell then uses
 * lad_profile[y] of lbm_create), else lbm_forest_code(h, y, y_m): bits 0-9 y = cells above the
 * forest base, bits 10-19 h = forest height in cells, bits 20-31 y_m = height of the LAD maximum in
 * eighths of a cell (0 = constant LAD).  The cell's LAD is a_fm * shape((y+1/2)/h, y_m/h) of
 * Eqs. 14-15 (a_fm when y_m = 0).  At most 255 distinct codes; the device keeps one byte per cell
 * (read only in rows that hold coded cells) and a table of C_D a_f.  NULL removes the codes.
 * LBM_EINVAL without LBM_SOLID_MASK.  Call after lbm_bind, at any time; synchronises the stream. */
int lbm_set_solid(lbm_t *h, const uint8_t *solid_host);
int lbm_set_forest_codes(lbm_t *h, const uint32_t *code_host, double a_fm);
uint32_t lbm_forest_code(int h, int y, double y_m);

/* Attach the caller-owned device workspace and stream; uploads the per-row tables.
 * Errors: LBM_ENOMEM (bytes < lbm_workspace_bytes or pointer not 256-B aligned), LBM_ECUDA. */
int lbm_bind(lbm_t *h, void *dev_workspace, size_t bytes, void *cuda_stream);

/* Momentum reference of the collision arithmetic: jx_ref_host, host,
 * ny doubles, an estimate of the mean streamwise momentum rho*u_x of each row (NULL = 0).  The
 * kernels evaluate the momentum channel of the collision about it, which removes the rounding of
 * the mean flow from the fp32 result; it never changes what is computed in exact arithmetic, any
 * finite profile is valid, and the closer it is to the flow the smaller the rounding error.
 * lbm_init installs the synthetic initial profile; lbm_set_macros* and lbm_set_state leave the
 * reference as it is.  lbm_get_reference_profile returns the profile in use (as rounded by the
 * library; setting it again reproduces it exactly), so that a checkpoint of lbm_get_state + lbm_time
 * + this profile restarts a run bit for bit.  Call after lbm_bind; both synchronise the stream. */
int lbm_set_reference_profile(lbm_t *h, const double *jx_ref_host);
int lbm_get_reference_profile(lbm_t *h, double *jx_ref_host);

/* Choose the synthetic initial field used by lbm_init (R16): rho = 1,
 * u = U(y_j) e_x + noise_frac*U_ref*(2r-1) per component, r = rand01(seed, 3*cell+comp). */
int lbm_set_init(lbm_t *h, int kind, double U_ref, double noise_frac);

/* State 0: f = f_eq(1, u_init) (Eq. 3; R17); t = 0; statistics cleared.  Async on the stream. */
int lbm_init(lbm_t *h, uint64_t seed);

/* State 0 from caller fields: f = f_eq(rho, u).  rho: [nz][ny][nx] fp32, u: [3][nz][ny][nx] fp32.
 * _dev: device pointers (read asynchronously on the stream).  _host: host pointers, copied
 * through the workspace staging area (pinned memory makes the copies asynchronous); returns
 * after the last copy has been consumed. */
int lbm_set_macros(lbm_t *h, const float *rho_dev, const float *u_dev);
int lbm_set_macros_host(lbm_t *h, const float *rho_host, const float *u_host);

/* Advance n >= 0 time steps: one fused kernel launch per step (stream, moments, drag,
 * Smagorinsky tau, Guo-forced BGK collision, boundary links, store; plus the fused stage-1
 * plane sums and the stage-2 reduction kernel on sampled steps).  Asynchronous. */
int lbm_step(lbm_t *h, int n);

/* z-slab decomposition (LBM_Z_HALO; "only information from directly adjacent
 * points is required").  The handle is created with nz = nz_local + 2.  After
 * lbm_init / lbm_set_macros* and after every lbm_step(1) the caller exchanges the two faces with
 * its z neighbours: lbm_halo_pack(side, buf) copies the five populations leaving through the low
 * (side 0) or high (side 1) face into the device buffer [5][ny][nx] fp32; the neighbour passes the
 * buffer it received to lbm_halo_unpack(side, buf), side = the side of ITS OWN slab the data enters
 * through.  Where the five populations sit depends on the storage scheme and the time parity, and
 * the library knows (two-lattice: c_z = -1 of plane 1 / c_z = +1 of plane nz-2 leave and land in
 * the neighbour's ghost planes; single array at odd t: the same planes, opposite slot sets; single
 * array at even t: what leaves has been pushed into the ghost planes and lands in the neighbour's
 * boundary plane, except where the destination cell bounced its own population off a wall face or
 * a solid cell).  The caller only has to keep all slabs of a lattice on the same storage scheme.
 * All asynchronous on the bound stream.
 * lbm_set_z_slab tells the synthetic initial field where the slab sits: local plane 0 (the low
 * ghost) is global plane z_first - 1 of nz_global (periodic).  Statistics and lbm_get_macros
 * cover the interior planes (ghost-plane entries of lbm_get_macros are meaningless); plane
 * averages divide by nx*(nz-2).  To combine slabs, sum lbm_stats_read_raw over the ranks and
 * pass the sums to lbm_stats_from_raw (a slab never uses an accumulation centre). */
int lbm_set_z_slab(lbm_t *h, int z_first, int nz_global);
int lbm_halo_bytes(const lbm_t *h, size_t *bytes);
int lbm_halo_pack(lbm_t *h, int side, float *buf_dev);
int lbm_halo_unpack(lbm_t *h, int side, const float *buf_dev);

/* One time step of a z slab with the halo exchange overlapped by the interior update (what
 * lbm_step(1) + pack + exchange + unpack do one after the other):
 *   lbm_step_slab_begin  updates the two boundary planes (1 and nz-2), packs the faces of the new
 *                        state into send_lo_dev / send_hi_dev ([5][ny][nx] fp32 each, as
 *                        lbm_halo_pack side 0 / 1), records packed_event (a cudaEvent_t passed as
 *                        void*, may be NULL) on the bound stream, then launches the update of the
 *                        interior planes.  Asynchronous.
 *   the caller           makes its communication stream wait for packed_event, sends send_hi to
 *                        the upper and send_lo to the lower ring neighbour, receives the lower
 *                        neighbour's high face into recv_lo and the upper neighbour's low face
 *                        into recv_hi, and records ready_event there: the transfer runs while the
 *                        interior planes are being updated.
 *   lbm_step_slab_end    makes the bound stream wait for ready_event (NULL = no wait), unpacks the
 *                        two buffers into the new state (ghost or boundary planes), runs the statistics
 *                        stage 2 of a sampled step and advances lbm_time.  Asynchronous.
 * Results are bit-identical to the sequential form.  LBM_ESTATE if the calls do not alternate;
 * LBM_EINVAL without LBM_Z_HALO. */
int lbm_step_slab_begin(lbm_t *h, float *send_lo_dev, float *send_hi_dev, void *packed_event);
int lbm_step_slab_end(lbm_t *h, const float *recv_lo_dev, const float *recv_hi_dev, void *ready_event);

/* Raw running sums behind lbm_stats_read, for combining slabs: out_host [ny][LBM_NSTAT] doubles of
 * sum(u-u0), sum(v-v0), sum(w-w0), the six centred second-moment sums and sum(rho) over the
 * samples and cells seen so far (column 9 holds sum(rho)); centre_host [ny][3] doubles = (u0, v0, w0) per row (may be NULL);
 * *count = samples x contributing cells per plane (may be NULL).  Synchronises the stream. */
int lbm_stats_read_raw(lbm_t *h, double *out_host, double *centre_host, double *count);
/* Host helper: the [ny][LBM_NSTAT] table of lbm_stats_read from raw sums (column 9 = sum of rho),
 * an optional centre [ny][3] and the total count; count <= 0 gives zeros. */
int lbm_stats_from_raw(const double *raw_host, const double *centre_host, int ny, double count, double *out_host);

/* CUDA graphs for launch-bound lattices: with graphs on, lbm_step(n) replays blocks of about 32
 * time steps as one captured graph of the same kernel launches (bit-identical results) and runs
 * the remainder directly.  mode 0 off, 1 on, 2 auto (default: on for lattices of at most 2^22
 * cells).  Not used while kernel timing is on or while the caller is capturing the stream. */
int lbm_set_graphs(lbm_t *h, int mode);

/* Sample S_k of the current state (see "Time" above) into caller-owned buffers (layouts as in
 * lbm_set_macros).  Either pointer may be NULL.  _dev is asynchronous; _host synchronises. */
int lbm_get_macros(lbm_t *h, float *rho_dev, float *u_dev);
int lbm_get_macros_host(lbm_t *h, float *rho_host, float *u_host);

/* Statistics (L200, L251: time then x-z plane averaging; L210 needs <v'w'>).
 * lbm_stats_accumulate(every): every > 0 samples S_k on every every-th step taken by lbm_step
 * from now on (phase restarts), every == 0 switches sampling off.  Sums are kept.
 * lbm_stats_read: synchronises the stream; out is host [ny][LBM_NSTAT] doubles, columns
 *   <u>, <v>, <w>, <u'u'>, <v'v'>, <w'w'>, <u'v'>, <v'w'>, <u'w'>, <rho>,
 * with <a> = sum a / (nsamples nx nz) and <a'b'> = <ab> - <a><b> (R18); *nsamples may be NULL.
 * Returns LBM_EDIVERGED if a non-finite plane sum was seen.
 * lbm_stats_reset clears the sums and re-centres the accumulation about the current plane
 * means (a numerical shift only; results are unchanged up to rounding). */
int lbm_stats_accumulate(lbm_t *h, int every);
int lbm_stats_read(lbm_t *h, double *out_host, long long *nsamples);
int lbm_stats_reset(lbm_t *h);

/* Checkpoint / restart and tests: the populations in the plain "state k" representation
 * (post-collision, un-streamed), device [19][nz][ny][nx] fp32 of f_i - w_i in SPECIFICATION
 * numbering (velocity table below), whatever the storage mode and time parity hold internally.
 * lbm_get_state writes it (state unchanged).  lbm_set_state installs it as state t (t >= 0: the
 * step counter the state belongs to; its parity selects the AA representation / the lattice of
 * the two-lattice scheme), so that get_state -> set_state(., lbm_time) -> lbm_step continues a
 * run bit for bit, non-equilibrium part included (lbm_set_macros would discard it).  Solid cells
 * are stored as the rest state.  The statistics sums and the sampling phase are left as they are.
 * Both are asynchronous on the bound stream.  lbm_set_state: LBM_ESTATE before lbm_bind. */
int lbm_get_state(lbm_t *h, float *f_minus_w_dev);
int lbm_set_state(lbm_t *h, const float *f_minus_w_dev, long long t);

/* Divergence sentinel: the stage-2 statistics reduction and lbm_get_macros* set a
 * device flag when they meet a non-finite density.  lbm_stats_read, lbm_stats_read_raw and
 * lbm_get_macros_host return LBM_EDIVERGED once it is set; lbm_get_macros is asynchronous, so its
 * finding is reported by the next of those calls or by lbm_diverged, which synchronises the stream,
 * writes the flag (0/1) to *flag_host (may be NULL) and returns LBM_OK or LBM_EDIVERGED.  The flag
 * is cleared by lbm_init, lbm_set_macros* and lbm_stats_reset. */
int lbm_diverged(lbm_t *h, int *flag_host);

/* Number of steps taken since the last init / set_macros. */
long long lbm_time(const lbm_t *h);

/* Number of kernels this handle has launched since creation (bench.py's gpu_launches). */
long long lbm_launch_count(const lbm_t *h);

/* Tuning hook: override the thread-block shape (tx thread columns of V cells along x, ty rows;
 * tx*ty <= 256, tx divides nx/V with at most 8 blocks per row, ty divides ny*nz - or ny itself on
 * a handle that launches plane ranges: LBM_Z_HALO, or a lattice larger than the host-transfer
 * staging area, 256 MB unless the environment variable LBM_STAGING_BYTES says otherwise).  Call
 * before the first lbm_step.  LBM_EINVAL if the shape does not tile the lattice. */
int lbm_set_launch_shape(lbm_t *h, int tx, int ty);

/* Data-movement path of the step kernel.  mode is a bit mask of the step kinds whose stream-in goes
 * through the Tensor Memory Accelerator (lbm_tma.cuh: cp.async.bulk.tensor tile loads whose box
 * coordinates carry the link's row and slot, x shift taken in shared memory) instead of per-thread
 * 128-bit loads: bit 0 the AA even step, bit 1 the AA odd step, bit 2 the two-lattice pull step;
 * 0 = none.  rows = y rows per
 * 256-cell tile (1, 2 or 4, must divide ny; 0 = keep).  Both paths compute the same thing with the
 * same per-cell arithmetic.  Available with 4 cells per thread, nx % 256 == 0 and no solid mask
 * (LBM_EINVAL otherwise); the environment variable LBM_TMA="mode[,rows]" sets the default of new
 * handles.  Call before or between lbm_step calls. */
int lbm_set_tma(lbm_t *h, int mode, int rows);

/* Other SGS models ("the standard Smagorinsky model is used ... A future work is to
 * implement other SGS models"; reading R29).  Per-row tables generalise
 * Eq. 10 (L83) to nu_t = C_j (|S| - Sbar_j), never negative, i.e.
 *   tau_total = max( tau0, ( t_j + sqrt( t_j^2 + 18 sqrt(2) C_j Q^{1/2} / rho ) ) / 2 ),  t_j = tau0 - 3 C_j Sbar_j,
 * which covers the wall-damped Smagorinsky model (C_j from lbm_sgs_van_driest, Sbar = 0) and the
 * shear-improved Smagorinsky model (Sbar_j = magnitude of the mean shear, lbm_sgs_mean_shear of a
 * statistics table; the caller refreshes it as the mean profile develops).  csmag_row_host,
 * sbar_row_host: [ny] doubles, host memory, read during the call; NULL csmag_row = Cs^2 of
 * lbm_create on every row, NULL sbar_row = 0; both NULL restores the standard model.  Entries must be
 * finite and >= 0 (LBM_EINVAL).  Costs 0 bytes per cell (one 8-byte table entry per row); handles
 * with tables run the SGS variants of the step kernel, never the TMA path.  Call after lbm_bind
 * (LBM_ESTATE otherwise), before or between lbm_step calls. */
int lbm_set_sgs_rows(lbm_t *h, const double *csmag_row_host, const double *sbar_row_host);

/* van Driest wall damping of the Smagorinsky constant: csmag_row_out[j] = Cs^2 (1 - exp(-y+_j/A+))^2,
 * y+_j = d_j u_tau / nu, d_j = distance of the cell centre j + 1/2 to the bottom wall face (to the
 * nearer of the two wall faces with both_walls != 0); A+ is usually 26.  Host only. */
int lbm_sgs_van_driest(int ny, double Cs, double u_tau, double nu, double A_plus, int both_walls,
                       double *csmag_row_out);

/* Mean-shear magnitude of a statistics table ([ny][10] of lbm_stats_read, columns <u> and <w>):
 * sbar_row_out[j] = sqrt((d<u>/dy)^2 + (d<w>/dy)^2), central differences between cell centres; the
 * profile continues past a no-slip wall face as its odd image (bottom always; top with top_wall !=
 * 0) and past a free-slip / lid face as its even image.  Host only. */
int lbm_sgs_mean_shear(const double *stats_host, int ny, int top_wall, double *sbar_row_out);

/* Sweep direction of the step kernel.  mode 1 (default): consecutive time steps walk the rows of
 * the lattice in opposite directions, so that a step starts on the planes the previous step wrote
 * last and finds them in the L2 cache (on lattices of a few hundred MB a sizeable part of the
 * reads; on HBM-filling ones a per-mille effect).  mode 0: every step walks forward.  The order in
 * which cells are visited has no effect on the result (the update of a cell needs
 * the previous state of adjacent cells only): both modes are bit-identical.  The environment
 * variable LBM_SWEEP=0|1 sets the default of new handles.  LBM_EINVAL for any other mode. */
int lbm_set_sweep(lbm_t *h, int mode);

/* Measurement hook (bench.py "roofline"): with on != 0, lbm_step brackets every step-kernel
 * launch (the fused S1-S8 kernel only, not the stage-2 reduction) with a pair of CUDA events on
 * the bound stream, up to 4096 launches between reads.  lbm_kernel_timing_read synchronises the
 * stream, returns the summed device time of the bracketed launches in milliseconds and their
 * count, and clears the record.  Either output may be NULL. */
int lbm_set_kernel_timing(lbm_t *h, int on);
int lbm_kernel_timing_read(lbm_t *h, double *total_ms, long long *launches);

/* Plane statistics of ONE sample given as fields, with NO allocation of any kind (no cudaMalloc,
 * cudaFree, or allocating library call; no handle, no workspace) - for callers that cannot allocate:
 * code under CUDA graph capture, tight serving loops, harnesses that forbid it.  The two-stage
 * reduction of the statistics path (S8, S9) over x and z:
 *   rho_dev  device, [nz][ny][nx] fp32;  u_dev  device, [3][nz][ny][nx] fp32 (as lbm_get_macros writes)
 *   out_dev  device, [ny][LBM_NSTAT] doubles, the columns of lbm_stats_read for this one sample:
 *            <u>,<v>,<w>,<u'u'>,<v'v'>,<w'w'>,<u'v'>,<v'w'>,<u'w'>,<rho>, averages over the x-z plane
 * Asynchronous on cuda_stream (a cudaStream_t passed as void*, NULL = the default stream), on the
 * device that owns rho_dev.  The stage-1 row sums go through a scratch array of
 * LBM_STATIC_SCRATCH_BYTES that is part of the library image: every GPU that loads the library holds
 * it until the process exits.  Limit: 10 * 4 * ny * nz bytes must fit, i.e. ny*nz <= 419 430 rows
 * (and nz <= 65 535) - config 5 (384 x 1024) fits; LBM_EINVAL with the numbers in lbm_last_error()
 * otherwise.  Every call shares that array, which keeps the last call's contents (nothing needs to
 * start at zero: each call writes all it reads): calls that OVERLAP on the GPU - different streams,
 * different threads - race on it; calls on one stream are safe.  LBM_ECUDA on a CUDA error. */
#define LBM_STATIC_SCRATCH_BYTES (16 * 1024 * 1024)
int lbm_plane_stats_static(const float *rho_dev, const float *u_dev, int nx, int ny, int nz,
                           double *out_dev, void *cuda_stream);

/* Environment variables the library reads (measurement switches; none changes a result):
 *   LBM_STAGING_BYTES  size of the host-transfer staging area (default 256 MB), read at every call
 *   LBM_TMA="m[,r]"    default of lbm_set_tma for new handles (default 0: per-thread loads)
 *   LBM_SWEEP=0|1      default of lbm_set_sweep for new handles (default 1: alternating direction)
 *   LBM_GRID3=0|1      step launch on a 3-D grid (x chunk, row block, plane; default 1) or on the 1-D
 *                      grid whose index arithmetic needs two integer divisions; read once per process
 *   LBM_PDL=0|1        programmatic dependent launch of the step / statistics kernels (default 1);
 *                      read once per process
 *   LBM_WPART=0|1      per-warp statistics partials for every handle, not only geometry handles
 *                      (default 0); read once per process
 * DESIGN.md "Kernels" and profiles/r02_README.md give the A/B numbers behind the defaults. */

/* Name of the kernel variant lbm_step uses, e.g. "aa/v4/tx384x1" (static string per handle). */
const char *lbm_variant(const lbm_t *h);

void lbm_destroy(lbm_t *h);

const char *lbm_last_error(void);

/* Host helpers (no CUDA): leaf-area-density table of Eqs. 14-15 (L105-115; R14):
 * a_j = LAI * s(eta_j) / sum_k s(eta_k) for j < h, 0 above, eta_j = (j+1/2)/h,
 * s(eta) = r^n exp[n(1-r)], r = (1-eta_m)/(1-eta), n = 6 (eta < eta_m) or 1/2. */
int lbm_lad_profile(int h, int ny, double LAI, double eta_m, double *out_host);
/* The same shape with the paper's own normalisation (Table II): a_j = a_fm * s(eta_j) for
 * j < h (case 2: a_fm = 0.38 per metre, eta_m = 0.7), or the constant a_j = a_fm when eta_m = 0
 * (case 1: 0.215 per metre); a_fm per lattice length. */
int lbm_lad_eq14(int h, int ny, double a_fm, double eta_m, double *out_host);

/* Host helpers (no CUDA) for the paper's normalised outputs, applied to
 * the [ny][LBM_NSTAT] table of lbm_stats_read.
 *   lbm_wall_friction_velocity   Eq. 16 (L179) inverted: u_tau = sqrt(F H / rho), F the streamwise
 *                                force density, H the channel half height (full height of a
 *                                half channel), all in lattice units.
 *   lbm_forest_friction_velocity L210: u_* = [<u'v'>^2 + <v'w'>^2]^(1/4) at y/h = 2; y = 2h is the
 *                                face between rows 2h-1 and 2h, so the two rows are averaged.
 *                                LBM_EINVAL unless 1 <= h and 2h < ny.
 *   lbm_stats_normalise          out[j][0..2] = <u_a>/u_ref (L200 "<u+> = <u>/u_tau");
 *                                out[j][3..5] = sqrt(max(<a'a'>, 0))/u_ref (the RMS components);
 *                                out[j][6..8] = <a'b'>/u_ref^2; out[j][9] = <rho>.  out may alias
 *                                stats.  LBM_EINVAL if u_ref <= 0.
 *   lbm_wall_units               y+_j = (j + 1/2) u_tau / nu for the ny cell centres. */
int lbm_wall_friction_velocity(double F, double H, double rho, double *u_tau);
int lbm_forest_friction_velocity(const double *stats_host, int ny, int h, double *u_star);
int lbm_stats_normalise(const double *stats_host, int ny, double u_ref, double *out_host);
int lbm_wall_units(int ny, double u_tau, double nu, double *yplus_host);

/* Counter-based uniform generator of the input recipe: splitmix64 output function of
 * seed + (ctr+1)*0x9E3779B97F4A7C15; rand01 = top 53 bits * 2^-53. */
uint64_t lbm_mix64(uint64_t seed, uint64_t ctr);

/* D3Q19 numbering used by every external layout:
 *  0:(0,0,0) | 1:(+,0,0) 2:(-,0,0) 3:(0,+,0) 4:(0,-,0) 5:(0,0,+) 6:(0,0,-) |
 *  7:(+,+,0) 8:(-,-,0) 9:(+,-,0) 10:(-,+,0) 11:(+,0,+) 12:(-,0,-) 13:(+,0,-) 14:(-,0,+)
 *  15:(0,+,+) 16:(0,-,-) 17:(0,+,-) 18:(0,-,+);  w = 1/3, 1/18 (1-6), 1/36 (7-18). */

#ifdef __cplusplus
}
#endif
#endif /* LBM_B200_H */
