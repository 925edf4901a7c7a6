/* mfc_b200.h — C ABI of the B200-native hot path of MFC 5.0's method (arxiv 2503.07953).
 *
 * The library evaluates the finite-volume right-hand side of the 5-equation (Allaire) diffuse-interface
 * model with stiffened-gas EOS — conservative->primitive conversion, WENO5-JS reconstruction of the
 * primitives, HLLC fluxes, flux divergence and the alpha_i div(u) source — and advances it by SSP-RK3.
 * Every step runs in hand-written fp64 CUDA kernels for sm_100a; there is NO CPU fallback: if no CUDA
 * device is usable every call returns MFC_ERR_CUDA.  Options of mfc_params beyond that path: mapped or
 * WENO-Z weights (weno), the Kapila K div(u) term (model), the viscous stress (eta); and MFC_BC_HALO with
 * mfc_set_halo / mfc_pack_halo / mfc_rk3_stage(_parts) for slabs of one domain on several GPUs.
 *
 * Citations are PAPER.md lines (section / equation).  Readings of points the paper leaves open carry the
 * A-numbers of DESIGN.md §3.
 *
 * DATA LAYOUT (all state arrays q, w, rhs): dense fp64, structure of arrays, interior cells only (no
 * ghost cells in memory), x fastest:
 *     idx(v,i,j,k) = ((v*n[2] + k)*n[1] + j)*n[0] + i,        v = 0..neq-1,  neq = 2*N + D + 1
 * (N fluids, D dimensions; "two advected species (8 PDEs)" in 3D).  Variable slots, the same
 * for conservative q and primitive w (PAPER.md:165 lists them in this order):
 *     [0,N)        alpha_i rho_i                      (both q and w)
 *     [N,N+D)      rho u_d      in q,   u_d  in w
 *     N+D          E = rho e + 1/2 rho |u|^2 (per volume, A1) in q,   p  in w
 *     (N+D,2N+D]   alpha_i                            (both q and w)
 *
 * OWNERSHIP: the caller owns q, w, rhs.  "device" pointers are CUDA device pointers valid on the
 * handle's device (e.g. torch.Tensor.data_ptr()), 8-byte aligned; "host" pointers are ordinary host
 * memory (pinned memory makes the *_host calls faster but is not required).  The handle owns its scratch
 * (two state-sized arrays, D cell-sized arrays of velocities when eta > 0, a few bytes of reduction/flag
 * storage) and never frees caller memory.
 *
 * STREAMS: every kernel is enqueued on the stream given at mfc_init_grid (NULL = the legacy default
 * stream).  Calls marked "async" return after enqueueing.  Calls marked "syncs" wait for that stream.
 *
 * ERRORS: every call returns an mfc_status, never throws or aborts.  Argument errors are detected
 * synchronously and leave all buffers untouched.  CUDA launch errors are returned by the call that saw
 * them.  A non-physical state met by a kernel (rho <= 0 or c^2 <= 0 or NaN at a cell or a face, A19) sets
 * a sticky flag in the handle that mfc_check / mfc_cfl_dt report as MFC_ERR_NONPHYSICAL (results are then
 * whatever IEEE arithmetic gave; nothing is floored silently).  mfc_last_error() gives a thread-local text.
 *
 * THREADS: one handle may be used by one host thread at a time.
 */
#ifndef MFC_B200_H
#define MFC_B200_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mfc_grid mfc_grid; /* opaque, library-owned */

typedef enum {
  MFC_OK = 0,
  MFC_ERR_ARG = 1,
  MFC_ERR_ALLOC = 2,
  MFC_ERR_CUDA = 3,
  MFC_ERR_NONPHYSICAL = 4
} mfc_status;

/* Ghost-cell ("buffer region") boundary conditions, PAPER.md:203 (§3.3).  Extrapolation is the paper's
 * first-order extrapolation (ghost = nearest interior cell); periodic is required by BASELINE.json
 * (the paper's Taylor-Green case, implies it).  Periodic must be set on both ends. */
typedef enum { MFC_BC_PERIODIC = 0, MFC_BC_EXTRAP = 1, MFC_BC_HALO = 2 } mfc_bc;
/* MFC_BC_HALO (slab decomposition, the paper's "buffer regions ... populated through message passing", PAPER.md:203,
 * 762-770): allowed on either end of the LAST direction of a 2-D or 3-D grid.  The three ghost layers beyond that
 * end are read from an array the caller fills before every RHS evaluation (mfc_set_halo). */

/* Nonlinear weights of the fifth-order WENO reconstruction.  JS: alpha_r = d_r/(beta_r+eps)^2
 * (the weights BASELINE.json names).  M: the JS weights passed through the map of Henrick et al. and
 * renormalised ("mapped weights", PAPER.md:165 — the paper's default).  Z: alpha_r = d_r (1 + tau/(beta_r+eps)),
 * tau = |beta_0 - beta_2| (PAPER.md:562-566 with q = 1). */
typedef enum { MFC_WENO_JS = 0, MFC_WENO_M = 1, MFC_WENO_Z = 2 } mfc_weno;

/* Volume-fraction equation: d(alpha_i)/dt + u.grad(alpha_i) = K_i div(u).  ALLAIRE: K_i = 0 ("for some
 * problems K div(u) is not necessary, and the model reduces to that of Allaire et al.", PAPER.md:86 — what
 * BASELINE.json names).  KAPILA: two fluids, K_1 = K of eq. (5) (numerator rho_2 c_2^2 - rho_1 c_1^2),
 * K_2 = -K, with the cell-centre p and alpha_i and the face velocities of the Riemann solver. */
typedef enum { MFC_MODEL_ALLAIRE = 0, MFC_MODEL_KAPILA = 1 } mfc_model;

#define MFC_MAX_FLUIDS 3

typedef struct {
  int ndim;              /* D = 1..3 */
  int n[3];              /* cells per direction; n[d] must be 1 for d >= ndim */
  double dx[3];          /* uniform spacing per direction (> 0); ignored for d >= ndim */
  int nfluids;           /* N = 1..MFC_MAX_FLUIDS */
  const double *gamma;   /* host, N values: gamma_i   of e_i = (p + gamma_i pi_inf_i)/((gamma_i-1) rho_i) */
  const double *pi_inf;  /* host, N values: pi_inf_i; both copied at init */
  int bc_lo[3], bc_hi[3];/* mfc_bc per direction and end */
  double weno_eps;       /* epsilon of the WENO weights, PAPER.md:163/566 (A4); >= 1e-75 (the kernels evaluate the weights
                          * in product form, whose smallest term is (4 eps)^4) */
  double alpha_floor;    /* volume-fraction floor of the RK-stage clamp (A10) */
  int clamp;             /* 0: no clamp; 1: apply A10 after every RK stage */
  int weno;              /* mfc_weno: nonlinear weights of the reconstruction; 0 = MFC_WENO_JS */
  int model;             /* mfc_model: 0 = MFC_MODEL_ALLAIRE; MFC_MODEL_KAPILA needs nfluids == 2 */
  double eta;            /* uniform shear viscosity of the viscous stress T = 2 eta (D - tr(D) I/3), PAPER.md:63-67 (eqs. 1-2),
                          * in the momentum and energy equations; second-order central differences at the faces (A22).
                          * 0 = inviscid (BASELINE.json).  With MFC_BC_HALO the stencil reads the velocities of the ghost
                          * layer from the halo arrays. */
  int device;            /* CUDA device ordinal */
  void *stream;          /* cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default */
} mfc_params;

/* Create a handle: validates p, selects the <D,N> kernel instantiation, allocates scratch on p->device.
 * Uniform Cartesian grid of PAPER.md:131-141 (eq. 9-10).  Returns MFC_ERR_ARG / MFC_ERR_ALLOC / MFC_ERR_CUDA. */
mfc_status mfc_init_grid(const mfc_params *p, mfc_grid **out);

/* Syncs the stream, frees the handle and its scratch.  NULL is accepted. */
mfc_status mfc_free_grid(mfc_grid *g);

/* neq = 2N + D + 1; cells = n[0]*n[1]*n[2].  Return -1 for a NULL handle. */
int mfc_num_eqns(const mfc_grid *g);
long long mfc_num_cells(const mfc_grid *g);

/* w = primitives of q, cell by cell (eq.(4), 117, 165; O2):
 *   rho = sum alpha_i rho_i, u = rho u / rho, Gamma = sum alpha_i/(gamma_i-1),
 *   Pi = sum alpha_i gamma_i pi_inf_i/(gamma_i-1),  p = ((E - Pi) - 1/2 rho |u|^2)/Gamma.
 * q, w: device, neq*cells doubles; may alias.  async. */
mfc_status mfc_prim_from_cons(mfc_grid *g, const double *q, double *w);

/* rhs = L(q): eq.(10) with WENO5-JS reconstruction of the primitives,
 * the HLLC flux (wave speeds 653-654, S* 664, rho* 668), the face-velocity divergence
 * for the alpha_i div(u) term and ghost cells by index mapping.
 * q, rhs: device, neq*cells doubles, must not alias; rhs is overwritten.  async. */
mfc_status mfc_rhs(mfc_grid *g, const double *q, double *rhs);

/* As mfc_rhs but only the directions whose bit is set in dir_mask (bit d = direction d) contribute;
 * cells keep 0 from the other directions.  dir_mask must be 1..7 (else MFC_ERR_ARG).  The viscous rates (eta > 0) are part
 * of the result only for dir_mask == 7, whatever the number of dimensions; on a handle with eta > 0 any other mask that
 * covers all of the grid's directions (3 in 2-D, 1 in 1-D, ...) is refused with MFC_ERR_ARG rather than answered without
 * them.  Exists so that each directional sweep can be tested alone. */
mfc_status mfc_rhs_dirs(mfc_grid *g, const double *q, double *rhs, int dir_mask);

/* One SSP-RK3 step of size dt (the three-stage formula), in place on q, with the A10
 * clamp after each stage when enabled.  q: device.  Uses the handle's scratch.  async. */
mfc_status mfc_rk3_step(mfc_grid *g, double *q, double dt);

/* nsteps RK3 steps with a fixed dt (one call, same arithmetic as nsteps calls of mfc_rk3_step).  async. */
mfc_status mfc_rk3_steps(mfc_grid *g, double *q, double dt, int nsteps);

/* Slab decomposition along the last direction (one handle per slab, one process per GPU).
 * mfc_set_halo: device arrays of the ghost layers beyond the low / high end, each neq*3*plane doubles laid out
 *   [v][layer][plane], plane = cells / n[ndim-1] in the grid's own order, layer l = 0..2 <-> logical cells -3+l (low end)
 *   and n+l (high end).  Caller-owned, must stay valid and hold the neighbour's data whenever a sweep runs; an end
 *   without MFC_BC_HALO may pass NULL.
 * mfc_rk3_stage: stage s = 1, 2, 3 of the RK3 step alone (mfc_rk3_step == the three in order).  With halos the caller
 *   refreshes them from the state the stage sweeps before each stage; mfc_stage_input returns that array
 *   (stage 1: q itself; stages 2, 3: the handle's stage state), neq*cells doubles, device.  async.
 * mfc_rk3_step(s), mfc_advance and the *_host calls refuse a handle with MFC_BC_HALO (they cannot refresh halos).
 * mfc_pack_halo: copies the three layers next to the low end (cells 0..2 of the last direction) of that same array into
 *   send_lo and the three next to the high end (cells n-3..n-1) into send_hi, both [v][layer][plane], device, either may
 *   be NULL.  What a slab packs as send_lo is its lower neighbour's halo_hi; send_hi is the upper neighbour's halo_lo.
 *   async on the handle's stream. */
mfc_status mfc_set_halo(mfc_grid *g, const double *halo_lo, const double *halo_hi);
mfc_status mfc_pack_halo(mfc_grid *g, const double *q, int stage, double *send_lo, double *send_hi);
mfc_status mfc_rk3_stage(mfc_grid *g, double *q, double dt, int stage);
/* The same stage in two parts, so that the halo exchange can run while the first part computes: parts = 1 launches the
 * sweeps of the directions before the last (they read no ghost layer of the last direction), parts = 2 the sweep of the
 * last direction with the RK combination and clamp (it needs the halos), parts = 3 both (== mfc_rk3_stage).  Call part 1
 * before part 2, on the same q and dt.  In 1-D part 1 is empty; with eta > 0 on a handle with MFC_BC_HALO too (the viscous
 * stencil reads the ghost layer of the last direction), and part 2 is then the whole stage. */
mfc_status mfc_rk3_stage_parts(mfc_grid *g, double *q, double dt, int stage, int parts);
mfc_status mfc_stage_input(mfc_grid *g, const double *q, int stage, const double **state_out);

/* dt = cfl / max_cells sum_d (|u_d| + c)/dx_d  with the frozen-alpha mixture sound speed
 * c^2 = ((Gamma+1) p + Pi)/(Gamma rho)  (A5, A9; not in the paper — BASELINE.json asks for it).
 * q: device; dt_out: HOST pointer to one double.  syncs; also reports the sticky non-physical flag. */
mfc_status mfc_cfl_dt(mfc_grid *g, const double *q, double cfl, double *dt_out);

/* The same CFL time step for callers that must not allocate: no handle, no cudaMalloc / cudaFree /
 * cudaMallocHost, nothing that grows the CUDA heap.  Meant for code that runs where device memory is
 * not ours to take: a solver plugged into an application whose memory pool already owns all of HBM
 * (another cudaMalloc fails or fragments the pool), a step function called from inside a latency-critical
 * loop where an allocation is an implicit device-wide synchronisation, or a host that forbids allocation
 * after start-up.  Every other call in this header needs an mfc_grid, and mfc_init_grid allocates.
 *
 * Only ndim, n, dx, nfluids, gamma, pi_inf, device and stream of *p are read (validated as in
 * mfc_init_grid); the other fields are ignored.
 *   q              device, neq*cells doubles, conservative state in the layout above (input, untouched)
 *   cfl            CFL number
 *   dt_out         DEVICE pointer to one double: receives cfl / max_cells sum_d (|u_d| + c)/dx_d, the same
 *                  IEEE operations as mfc_cfl_dt, so the two agree bit for bit
 *   nonphysical_out DEVICE pointer to one int, may be NULL: receives 1 if some cell had rho <= 0 or
 *                  c^2 <= 0 or NaN (A19), else 0 — there is no handle to keep a sticky flag in
 * async on p->stream; it never synchronises, which is why both results stay on the device.
 *
 * SCRATCH: the per-block partial maxima and the completion counter live in one array that is part of the
 * library image, MFC_STATIC_SCRATCH_BYTES (129 KiB) on every GPU that loads the library, held until the
 * process exits.  A block reduces MFC_STATIC_CELLS_PER_BLOCK cells and there is room for
 * MFC_STATIC_MAX_BLOCKS partial results, so grids of more than MFC_STATIC_MAX_CELLS = 2^25 cells
 * (256^3 fits, 512^3 does not) are refused with MFC_ERR_ARG and a text saying so; nothing is launched.
 * The array is shared by every call in the process and keeps what the last call left there.  The call
 * clears the counter and flag words it depends on before launching, so a call that follows an aborted
 * one still starts clean — but two calls whose kernels overlap on one GPU (different streams, or
 * different host threads) race on it and may both return garbage.  Serialise them.
 *
 * FIRST CALL on each device looks up the device address of that array (one cudaGetSymbolAddress with the
 * device current, cached per device afterwards).  The lookup is not a stream operation, so make the
 * first call on a device outside of any stream capture. */
#define MFC_STATIC_CELLS_PER_BLOCK 2048
#define MFC_STATIC_MAX_BLOCKS 16384
#define MFC_STATIC_MAX_CELLS (1LL * MFC_STATIC_CELLS_PER_BLOCK * MFC_STATIC_MAX_BLOCKS)
#define MFC_STATIC_SCRATCH_BYTES (8 * MFC_STATIC_MAX_BLOCKS + 1024)
mfc_status mfc_cfl_dt_static(const mfc_params *p, const double *q, double cfl, double *dt_out, int *nonphysical_out);

/* Syncs and returns MFC_ERR_NONPHYSICAL if any kernel since the last mfc_check flagged a non-physical
 * state (clears the flag), MFC_ERR_CUDA on an asynchronous CUDA error, else MFC_OK. */
mfc_status mfc_check(mfc_grid *g);

/* End-to-end forms over HOST buffers (the calls bench.py's "e2e" leg times): copy q_host to the handle's
 * device staging (allocated on first use), run, copy the result back, sync.
 *   mfc_rhs_host:        rhs_host = L(q_host)
 *   mfc_rk3_steps_host:  q_host advanced in place by nsteps steps of size dt */
mfc_status mfc_rhs_host(mfc_grid *g, const double *q_host, double *rhs_host);
mfc_status mfc_rk3_steps_host(mfc_grid *g, double *q_host, double dt, int nsteps);

/* Adaptive stepping, all on the device timeline: nsteps times { dt = CFL step of the current state (as
 * mfc_cfl_dt); one RK3 step of size dt }.  *t_elapsed_host (HOST, may be NULL) receives the sum of the dt.
 * dt never leaves the device: a one-thread kernel turns the reduction's maximum into dt and adds it to the elapsed time,
 * the RK stages read it from device memory — same kernels and IEEE arithmetic as the caller's own loop of mfc_cfl_dt +
 * mfc_rk3_step (bit-identical states and elapsed time), without a host round trip per step.  Both calls synchronise once,
 * at the end, and then report the sticky non-physical flag (a state that turns non-physical in step k is still stepped to
 * the end).  mfc_advance: q device.  mfc_advance_host: q_host HOST, copied in before and out after the nsteps steps. */
/* On grids of at most 2^18 cells (launch-bound: BASELINE.json configs 1 and 2) both calls replay a CUDA graph of two steps
 * — one graph launch instead of 22 kernel launches — captured on the third step of a handle and re-captured when q or cfl
 * change; same kernels, arguments and order, hence the same bits.  mfc_set_step_graph(g, 0) turns that off (on by default;
 * it is also off while profiling is on).  The replay runs on a stream of the handle's own, ordered behind and before the
 * handle's stream by events. */
mfc_status mfc_advance(mfc_grid *g, double *q, double cfl, int nsteps, double *t_elapsed_host);
mfc_status mfc_advance_host(mfc_grid *g, double *q_host, double cfl, int nsteps, double *t_elapsed_host);

/* Per-kernel device timing for the benchmark's roofline line.  While profiling is on, every kernel launch
 * of this handle is bracketed by CUDA events on the handle's stream.  mfc_get_profile syncs and returns,
 * for one kernel class, the summed device time in ms and the number of launches since mfc_set_profiling(g,1).
 * Kernel classes: */
enum { MFC_K_PRIM = 0, MFC_K_SWEEP_X = 1, MFC_K_SWEEP_Y = 2, MFC_K_SWEEP_Z = 3, MFC_K_RK = 4, MFC_K_CFL = 5, MFC_K_COUNT = 6 };
mfc_status mfc_set_profiling(mfc_grid *g, int on); /* on = 1 also clears the accumulated profile */
mfc_status mfc_get_profile(mfc_grid *g, int kernel_class, double *total_ms_host, long long *launches_host);

/* Unit-level entry points of the two device functions every sweep kernel is built from (used by the parity
 * tests to compare them one by one with the oracle's weno5_js / hllc_face; not needed by applications).
 *   mfc_weno5_values: count stencils of 5 doubles each (stencil-major: s[5*t + k] = w_{i-2+k}) ->
 *       left[t]  = left-biased value at i+1/2, right[t] = right-biased value at i-1/2
 *   mfc_hllc_faces: count faces with reconstructed primitives wL, wR (face-major, neq values per face) ->
 *       F (face-major, neq per face) and uf[count]; dir = face normal
 * All pointers device; async. */
mfc_status mfc_weno5_values(mfc_grid *g, const double *stencils, long long count, double *left, double *right);
mfc_status mfc_hllc_faces(mfc_grid *g, int dir, const double *wL, const double *wR, long long count, double *F, double *uf);

/* Unit-level entry point of the square root of a ratio the Riemann solver uses for the face sound speed,
 * c = sqrt(cn / (Gamma rho)) (A5): out[t] = a[t] * rsqrt(a[t] b[t]) refined once, as in the sweeps, and (seed_out not NULL)
 * the raw hardware rsqrt(a[t] b[t]) the refinement starts from.  Valid where the PRODUCT a b is a normal double that
 * neither overflows nor is flushed to zero (about 1e-307 < a b < 1e308; for the sound speed a b ~ p Gamma rho, 1e3..1e14
 * in SI units); a product that underflows makes the sweeps flag the face as non-physical, one that overflows gives 0.
 * All pointers device, count doubles each; async. */
mfc_status mfc_sqrt_ratio_values(mfc_grid *g, const double *a, const double *b, long long count, double *out, double *seed_out);

/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
long long mfc_launch_count(const mfc_grid *g);

/* Measurement aid for the roofline (no part of the path): sustained vector-FP64 throughput of `device` in TFLOP/s
 * (2 flop per DFMA) from register-resident DFMA chains on all SMs — with two loop-invariant operands (the pipe's
 * issue rate) and with three distinct, changing register operands.  Host pointers; syncs. */
mfc_status mfc_measure_fp64(int device, void *stream, double *dfma_tflops_host, double *dfma3_tflops_host);

/* Tuning knob (benchmarks/tests only): cells per thread segment along the sweep direction, per direction;
 * 0 keeps the library's choice.  Results do not depend on it beyond round-off-free re-partitioning
 * (each face flux is computed from the same inputs wherever the segment boundaries fall). */
mfc_status mfc_set_segments(mfc_grid *g, int seg_x, int seg_y, int seg_z);

/* on = 0: mfc_advance / mfc_advance_host launch every kernel of every step themselves, whatever the grid size (see there). */
mfc_status mfc_set_step_graph(mfc_grid *g, int on);

/* Text of the last error on this host thread ("" if none). */
const char *mfc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MFC_B200_H */
