/* hydro.h -- C ABI of the B200 (sm_100a) unsplit patch-group fluid solver.
 *
 * Hot path of Schive, Zhang & Chiueh, "Directionally Unsplit Hydrodynamic Schemes with Hybrid
 * MPI/OpenMP/GPU Parallelization in AMR" (arXiv:1103.3373): the Riemann-solver-based,
 * directionally unsplit update of a batch of AMR patch groups.
 *
 *   - unit of work: a patch group = 2x2x2 patches of 8^3 cells = 16^3 interior cells, sent to the
 *     GPU together with its ghost zones (section 3.1; section 4.2);
 *   - the update: steps (1)-(5) of PAPER.md:39-44 (section 2): reconstruct + half-step face values,
 *     Riemann solve, transverse-flux correction + second Riemann solve (CTU), conservative update,
 *     store of the fluxes across patch boundaries;
 *   - options: schemes MHM / VL / CTU, PLM / PPM with four limiters on primitive
 *     or characteristic variables, exact / HLLE / HLLC / Roe solvers with the Roe
 *     failure fallback;
 *   - the evolution time-step (a CPU task in the paper) as a device reduction.
 *
 * The paper gives no formulas; the exact arithmetic is fixed by DESIGN.md ("Readings").
 *
 * Conventions
 *   variables   v = 0..4 : rho, rho*vx, rho*vy, rho*vz, E ; ideal gas E = P/(gamma-1) + rho|v|^2/2.
 *   layout      x fastest, structure of arrays per group, S = 16 + 2*nghost:
 *                 in       [Ng][5][S][S][S]            (z, y, x)
 *                 out      [Ng][5][16][16][16]
 *                 face_flux[Ng][9][5][16][16]          plane p = 3*d + s, d = 0,1,2 (x,y,z normal),
 *                                                       s = 0,1,2 <-> face index f = 0, 8, 16 (the
 *                                                       boundaries of the 8^3 patches); in-plane
 *                                                       order d=x:[k][j], d=y:[k][i], d=z:[j][i];
 *                                                       raw time-centred flux density (not x dt, area).
 *   ownership   every pointer is caller-owned; the library allocates nothing, frees nothing and
 *               keeps no state between calls (hydro_pipeline_* below owns only its own staging).
 *               Device pointers must be 16-byte aligned; in / out / face_flux must not overlap.
 *   async       device entry points only enqueue work on `stream` and return; no host sync.
 *   errors      0 = success; < 0 = argument error detected on the host before any launch
 *               (HYDRO_E_*); > 0 = cudaError_t of a failed launch.  Ng == 0 is a no-op returning 0.
 *               Numerical trouble (non-positive rho/P, Roe failure, Newton failure) is never an
 *               error code: it is counted in hydro_opts::status.
 *   no fallback there is no CPU path and no other backend.
 */
#ifndef HYDRO_H_
#define HYDRO_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define HYDRO_API __attribute__((visibility("default")))
#else
#define HYDRO_API
#endif

typedef struct CUstream_st* hydro_stream_t; /* == cudaStream_t; 0 = the legacy default stream */

enum { HYDRO_MHM = 0, HYDRO_VL = 1, HYDRO_CTU = 2 };                       /* scheme */
enum { HYDRO_EXACT = 0, HYDRO_HLLE = 1, HYDRO_HLLC = 2, HYDRO_ROE = 3 };   /* riemann */
enum { HYDRO_GMINMOD = 0, HYDRO_VANLEER = 1, HYDRO_VANALBADA = 2, HYDRO_HYBRID = 3 }; /* limiter PAPER.md:48 */
enum { HYDRO_PLM = 0, HYDRO_PPM = 1 };                                     /* recon */
/* kernel organisation (both compute the same update): staged = one phase per stage with global scratch (any
 * variant, any ghost width); fused = z-marching, every intermediate on chip, phase-crossing state in shared
 * memory (CTU, MHM and VL; two CTAs per SM where the tiles allow).  AUTO picks fused when it exists and its tiles fit. */
enum { HYDRO_IMPL_AUTO = 0, HYDRO_IMPL_STAGED = 1, HYDRO_IMPL_FUSED = 2 };

enum {
  HYDRO_OK = 0,
  HYDRO_E_ENUM = -1,      /* scheme / riemann / limiter / recon / roe_fallback / norm / impl out of range */
  HYDRO_E_COUNT = -2,     /* Ng < 0 */
  HYDRO_E_NULL = -3,      /* a required pointer is NULL */
  HYDRO_E_ALIGN = -4,     /* a device pointer is not 16-byte aligned */
  HYDRO_E_GHOST = -5,     /* nghost < hydro_min_ghost(scheme, recon), or > 8 */
  HYDRO_E_WORKSPACE = -6, /* staged path selected and workspace missing / smaller than one slot */
  HYDRO_E_VALUE = -7,     /* gamma <= 1, dh <= 0, dt < 0, minmod_coeff outside [1,2], negative floor, cfl <= 0 */
  HYDRO_E_NOFUSED = -8,   /* impl == HYDRO_IMPL_FUSED and no such kernel exists (or fits) for this variant */
  HYDRO_E_TOOBIG = -9     /* a size beyond the fixed maximum of an entry point that allocates nothing (hydro_rtvd_solve_noalloc_f64) */
};

typedef struct hydro_opts {      /* NULL => all defaults */
  int recon;            /* HYDRO_PLM (default) / HYDRO_PPM */
  int nghost;           /* ghost width of `in`; 0 => hydro_min_ghost(scheme, recon)                  */
  int char_limit;       /* 0 limit primitive variables (default), 1 characteristic */
  float minmod_coeff;   /* theta in [1,2] of the generalized minmod limiter; 0 => 1.5                */
  int roe_fallback;     /* solver used at a face where Roe fails: 0/1 HLLE, 2 HLLC, 3 exact PAPER.md:50 */
  double min_dens;      /* density floor, 0 => none (default)                                        */
  double min_pres;      /* pressure floor, 0 => none (default)                                       */
  long long* status;    /* device long long[3] or NULL; accumulated atomically:
                           [0] Roe failures, [1] non-positive rho or P seen by a conversion (the fp32 fused CTU kernel
                           with default options counts (thread, plane) pairs that met one, not single conversions:
                           non-zero exactly when the others are), [2] exact-solver vacuum / non-convergence   */
  void* workspace;      /* device scratch for the staged path (hydro_workspace_bytes); else NULL     */
  size_t workspace_bytes;
  int impl;             /* HYDRO_IMPL_AUTO: a fused z-marching kernel when one exists and fits, else staged */
  const void* max_speed;/* device scalar (float / double as the call) or NULL.  If set, the `dt` argument is
                           ignored and dt/dh = cfl / *max_speed is formed on the device, so that
                           hydro_dt -> hydro_solve stays asynchronous (no host read of the reduction)   */
  double cfl;           /* CFL number used with max_speed (> 0)                                       */
  void* next_max_speed; /* device scalar (float / double as the call) or NULL.  If set, it receives the hydro_dt reduction
                           (norm `next_norm`) of the UPDATED state `out`, formed inside the update (fused kernels) or by a
                           hydro_dt launch on `out` (staged kernel): the next step's max_speed without another pass
                           over the data.  Must not alias max_speed                                     */
  int next_norm;        /* 0 / 1 as in hydro_dt                                                         */
} hydro_opts;

/* One unsplit update of Ng patch groups.  in/out/face_flux: device pointers,
 * layouts above; face_flux may be NULL (step (5) skipped).  dt, dh, gamma: one value per call (a batch
 * belongs to one AMR level). */
HYDRO_API int hydro_solve_f32(const float* in, float* out, float* face_flux, int Ng, float dt, float dh, float gamma,
                    int scheme, int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream);
HYDRO_API int hydro_solve_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma,
                    int scheme, int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream);

/* Evolution time-step reduction: maximum over the INTERIOR cells of all groups of
 *   norm 0: max_d |v_d| + c        norm 1: sum_d |v_d| + 3 c ,   c = sqrt(gamma P / rho).
 * u has the layout of `in` with ghost width nghost (>= 0).  *max_speed (device scalar) is overwritten;
 * it is NaN if any interior cell has non-positive rho or P.  The caller forms dt = CFL*dh / *max_speed. */
HYDRO_API int hydro_dt_f32(const float* u, int Ng, int nghost, float gamma, int norm, float* max_speed, hydro_stream_t stream);
HYDRO_API int hydro_dt_f64(const double* u, int Ng, int nghost, double gamma, int norm, double* max_speed, hydro_stream_t stream);

/* Host-buffer entry points (the paper's asynchronous-copy pipeline: `nstreams`
 * CUDA streams, each cycling chunks of `groups_per_chunk` patch groups through H2D copy -> kernel ->
 * D2H copy so that transfers overlap the solver).  The pipeline object owns its device staging
 * buffers and streams; in/out/face_flux are HOST pointers (pinned memory gives real overlap) and the
 * call returns after all results are in `out` / `face_flux`.  opts->workspace/status/max_speed are
 * ignored; status counters, if wanted, are returned in status_host[3] (host, may be NULL).
 * max_speed_host (host scalar, may be NULL) receives the hydro_dt reduction (norm 0) of the UPDATED
 * state, computed chunk by chunk while the data is still on the device: the next step's dt. */
typedef struct hydro_pipeline hydro_pipeline;
HYDRO_API int hydro_pipeline_create(hydro_pipeline** p, int precision_bytes, int nghost, int groups_per_chunk, int nstreams);
HYDRO_API void hydro_pipeline_destroy(hydro_pipeline* p);
HYDRO_API int hydro_pipeline_solve_f32(hydro_pipeline* p, const float* in, float* out, float* face_flux, int Ng, float dt,
                             float dh, float gamma, int scheme, int riemann, int limiter, const hydro_opts* opts,
                             long long* status_host, float* max_speed_host);
HYDRO_API int hydro_pipeline_solve_f64(hydro_pipeline* p, const double* in, double* out, double* face_flux, int Ng, double dt,
                             double dh, double gamma, int scheme, int riemann, int limiter, const hydro_opts* opts,
                             long long* status_host, double* max_speed_host);

/* Device-side preparation / closing steps for UNIFORM grids (the paper does them on the CPU, where they
 * take up to 3x the GPU time).  grid: device [5][nz][ny][nx] (x fastest), nx, ny, nz multiples of 16; groups: device
 * [Ng][5][(16+2*nghost)^3] with Ng = (nx/16)(ny/16)(nz/16) and group n = (gz*(ny/16) + gy)*(nx/16) + gx.
 * hydro_gather_* copies every patch group with its ghost zones out of the grid; bc 0: periodic wrap, 1: outflow
 * (zero-gradient clamp) at the domain boundary.  hydro_scatter_* copies updated interiors out[Ng][5][16^3] back.
 * Pure copies (bit-exact), asynchronous on `stream`; pointers caller-owned, 16-byte aligned, not overlapping.
 * Errors: HYDRO_E_VALUE (a dimension not a multiple of 16), HYDRO_E_GHOST (nghost > 8), HYDRO_E_ENUM (bc). */
HYDRO_API int hydro_gather_f32(const float* grid, float* groups, int nx, int ny, int nz, int nghost, int bc, hydro_stream_t stream);
HYDRO_API int hydro_gather_f64(const double* grid, double* groups, int nx, int ny, int nz, int nghost, int bc, hydro_stream_t stream);
HYDRO_API int hydro_scatter_f32(const float* out, float* grid, int nx, int ny, int nz, hydro_stream_t stream);
HYDRO_API int hydro_scatter_f64(const double* out, double* grid, int nx, int ny, int nz, hydro_stream_t stream);

/* One update of a UNIFORM grid in one launch (no gather / scatter pass, no group buffers): the fused kernel fetches the
 * planes of every patch group from grid_in [5][nz][ny][nx] directly, ghost zones of width hydro_min_ghost() folded at the
 * domain boundary (bc 0 periodic, 1 outflow), and writes the updated cells to grid_out (same shape; must not be grid_in).
 * opts as in hydro_solve_* (nghost, workspace and impl ignored; face fluxes are not produced).  Available for every scheme
 * (MHM, VL, CTU), reconstruction, Riemann solver and limiter option; the one exception is VL with positivity floors
 * (min_dens / min_pres > 0), which returns HYDRO_E_NOFUSED: the caller then uses hydro_gather_* -> hydro_solve_* ->
 * hydro_scatter_*.  Results equal that three-call path bit for bit with the default options (van Leer limiter on
 * primitive variables, no floors) and to a few ulp otherwise. */
HYDRO_API int hydro_solve_grid_f32(const float* grid_in, float* grid_out, int nx, int ny, int nz, int bc, float dt, float dh,
                         float gamma, int scheme, int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream);
HYDRO_API int hydro_solve_grid_f64(const double* grid_in, double* grid_out, int nx, int ny, int nz, int bc, double dt, double dh,
                         double gamma, int scheme, int riemann, int limiter, const hydro_opts* opts, hydro_stream_t stream);

/* `steps` updates of a UNIFORM grid without leaving the device (the paper's preparation / solver / closing
 * cycle, with the evolution time-step of PAPER.md:137 formed on the device): hydro_dt of the start state once,
 * then per step dt = opts->cfl * dh / max_speed, the update, and the wave speed of the new state for the next step (fused into
 * the update, hydro_opts::next_max_speed).  Variants hydro_solve_grid_* covers run ONE launch per step between `grid` and a
 * second grid in `work` (unless opts->nghost is set, which asks for the group path); the others run hydro_gather -> hydro_solve -> hydro_scatter with the group buffers (and the staged
 * scratch, if that path is taken) in `work`.  grid: device [5][nz][ny][nx], updated in place.  opts: required; cfl > 0;
 * recon, nghost (0 = minimum), char_limit, floors, roe_fallback, status, impl as in hydro_solve_*; max_speed, next_max_speed,
 * workspace are ignored.  work: device scratch of hydro_advance_workspace_bytes(...), 256-byte aligned, caller-owned.
 * elapsed: device double or NULL; the sum of the steps' dt is ADDED to it (by a one-thread kernel on `stream`).
 * Asynchronous on `stream`, no host synchronisation, capturable in a CUDA graph.  Errors as hydro_solve_*, plus
 * HYDRO_E_COUNT (steps < 0), HYDRO_E_WORKSPACE (work too small), HYDRO_E_VALUE (opts NULL or cfl <= 0). */
HYDRO_API size_t hydro_advance_workspace_bytes(int nx, int ny, int nz, int precision_bytes, int scheme, int limiter, const hydro_opts* opts);
HYDRO_API int hydro_advance_f32(float* grid, int nx, int ny, int nz, int bc, int steps, float dh, float gamma, int scheme, int riemann,
                                int limiter, const hydro_opts* opts, void* work, size_t work_bytes, double* elapsed, hydro_stream_t stream);
HYDRO_API int hydro_advance_f64(double* grid, int nx, int ny, int nz, int bc, int steps, double dh, double gamma, int scheme, int riemann,
                                int limiter, const hydro_opts* opts, void* work, size_t work_bytes, double* elapsed, hydro_stream_t stream);

/* Consumer of face_flux: coarse-fine flux fix-up and fine -> coarse restriction after the fluid update of two adjacent AMR
 * levels (section 2 step 5: the stored fluxes are "only necessary in AMR"; section 4.3: the
 * "coarse-grid correction", a CPU task in the paper).  The paper gives no formula; reading S25 of DESIGN.md:
 *   - a refined coarse patch (8^3 coarse cells) is covered by exactly ONE fine patch group (16^3 fine cells), so the outer
 *     boundary planes of the fine group (face_flux planes p = 3 d + s, s = 0 or 2) coincide with the faces of the coarse patch,
 *     each coarse face being covered by 2 x 2 fine faces;
 *   - hydro_restrict_*: for every entry of map[n][5] = (fine_group, coarse_group, pi, pj, pk) the 8^3 coarse cells of
 *     coarse_out[coarse_group] starting at (pi, pj, pk) (each 0 or 8) become the means of their eight fine cells of
 *     fine_out[fine_group], summed ((x pairs) + (x pairs)) over y, then over z, times 1/8: bit-exact with the oracle;
 *   - hydro_fluxfix_*: for every entry of faces[n][7] = (fine_group, dir, fine_side, coarse_group, ci, cj, ck): the 8 x 8 layer of
 *     UNREFINED coarse cells of coarse_out[coarse_group] adjacent to the face -- (ci, cj, ck) is the first cell of the layer:
 *     along dir the layer index, in-plane a multiple of 8 -- is corrected by
 *         U += sigma (dt_c / dh_c) (F_c - ((f00 + f10) + (f01 + f11)) / 4),
 *     F_c = coarse_flux[coarse_group][3 dir + s] at the cell's face toward the fine group (s = (layer + 1) / 8 if the fine group
 *     lies above the layer, fine_side = 0: its LOWER boundary plane is the face; s = layer / 8 if below, fine_side = 1),
 *     f.. = the 2 x 2 fine fluxes of fine_flux[fine_group][3 dir + 2 fine_side], sigma = +1 (fine_side 0) or -1.  Contributions
 *     of several faces to one cell are added atomically (their order is not fixed: rounding-level only).
 *   - hydro_flux_accum_*: acc += w * face_flux over n elements (the dt-weighted time average of sub-cycled fine fluxes).
 * coarse_out / fine_out are the `out` arrays of hydro_solve_* of the two levels, coarse_flux / fine_flux their `face_flux`
 * arrays (raw flux densities); faces / map: device int arrays.  All pointers device, caller-owned, 16-byte aligned (int lists:
 * 4); asynchronous on `stream`.  Errors: HYDRO_E_COUNT (n < 0), HYDRO_E_NULL, HYDRO_E_ALIGN, HYDRO_E_VALUE (dh_c <= 0, dt_c < 0).
 * Index values are NOT range-checked (device data). */
HYDRO_API int hydro_fluxfix_f32(float* coarse_out, const float* coarse_flux, const float* fine_flux, const int* faces, int nfaces,
                                float dt_c, float dh_c, hydro_stream_t stream);
HYDRO_API int hydro_fluxfix_f64(double* coarse_out, const double* coarse_flux, const double* fine_flux, const int* faces, int nfaces,
                                double dt_c, double dh_c, hydro_stream_t stream);
HYDRO_API int hydro_restrict_f32(const float* fine_out, float* coarse_out, const int* map, int n, hydro_stream_t stream);
HYDRO_API int hydro_restrict_f64(const double* fine_out, double* coarse_out, const int* map, int n, hydro_stream_t stream);
HYDRO_API int hydro_flux_accum_f32(float* acc, const float* face_flux, long long n, float w, hydro_stream_t stream);
HYDRO_API int hydro_flux_accum_f64(double* acc, const double* face_flux, long long n, double w, hydro_stream_t stream);

/* The directionally SPLIT relaxing-TVD update: the scheme of the original GAMER ("RTVD; Jin & Xin
 * 1995 ... with directional splitting") that the paper times next to the unsplit schemes as the contrast with one-dimensional
 * stencils and low arithmetic intensity.  Same batch layouts as hydro_solve_* (in [Ng][5][S^3] with
 * nghost >= 3, out [Ng][5][16^3], face_flux [Ng][9][5][16 x 16] or NULL).  Reading S26 of DESIGN.md: every conserved variable is
 * split into right / left movers (c U +- F_d(U)) / 2 with the freezing speed c = |v_d| + c_s of its cell; one sweep = a
 * first-order predictor to dt/2 and a corrector with van-Leer-limited MUSCL fluxes of the movers evaluated at the predicted
 * state; one call = three sweeps with the same dt in the order x, y, z (order 0) or z, y, x (order 1; alternate them from step
 * to step).  face_flux receives the corrector flux of each direction's sweep at the faces f = 0, 8, 16 (the flux that sweep
 * used, so that the flux balance of hydro_solve_* holds).  opts: nghost (0 => 3), status ([1] counts non-positive rho / P),
 * max_speed + cfl (dt formed on the device), workspace + workspace_bytes: hydro_rtvd_workspace_bytes(Ng, precision)
 * (at least one slot of 5 x (22 x 22 x 16 + 22 x 16 x 16) elements; the kernel runs one CTA per slot) -- REQUIRED in fp64 and
 * for nghost > 3; fp32 with nghost == 3 keeps the whole padded group in shared memory and ignores it.  No Riemann solver, no
 * limiter choice, no floors.  Errors as hydro_solve_* (HYDRO_E_GHOST: nghost < 3; HYDRO_E_WORKSPACE; HYDRO_E_ENUM: order). */
HYDRO_API size_t hydro_rtvd_workspace_bytes(int Ng, int precision_bytes);
HYDRO_API int hydro_rtvd_solve_f32(const float* in, float* out, float* face_flux, int Ng, float dt, float dh, float gamma, int order,
                                   const hydro_opts* opts, hydro_stream_t stream);
HYDRO_API int hydro_rtvd_solve_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma, int order,
                                   const hydro_opts* opts, hydro_stream_t stream);

/* The directionally SPLIT weighted-average-flux update: the second split scheme the paper times next to the
 * unsplit ones ("the weighted average flux scheme (WAF; see Toro 2009)").  Reading S29 of DESIGN.md: TVD WAF with the
 * HLLC wave structure on piecewise-constant data -- at a face, F = (F_L + F_R)/2 - 1/2 sum_k sign(c_k) A_k (F(k+1) - F(k)) over the
 * waves S_L, S*, S_R of the HLLC solution, c_k = dt S_k / dh, A_k = 1 - (1 - |c_k|) B(r_k) with the van Leer limiter B of the ratio
 * of the upwind to the local jump across wave k (of the density; of the tangential momentum components themselves across the
 * contact); one call = three sweeps x, y, z (order 0) or z, y, x (order 1).  Arguments, layouts, workspace
 * (hydro_rtvd_workspace_bytes), face_flux planes, status and errors exactly as hydro_rtvd_solve_*; nghost >= 3 (the scheme
 * itself uses two of the ghost layers).  Needs max_k |c_k| <= 1: dt <= dh / hydro_dt's maximum speed. */
HYDRO_API int hydro_waf_solve_f32(const float* in, float* out, float* face_flux, int Ng, float dt, float dh, float gamma, int order,
                                  const hydro_opts* opts, hydro_stream_t stream);
HYDRO_API int hydro_waf_solve_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma, int order,
                                  const hydro_opts* opts, hydro_stream_t stream);

/* The same split relaxing-TVD update (reading S26) through an entry point that ALLOCATES NOTHING, for
 * callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it): fp64, ghost
 * width 3 (in [Ng][5][22^3]), the kernel of hydro_rtvd_solve_f64 with its scratch slots in a file-scope device array of the
 * library instead of a caller workspace: 32 slots = 17 121 280 bytes (16.3 MiB), which every GPU that loads the library holds
 * until exit.  The caller still passes in, out, face_flux (or NULL) and status (device long long[3] or NULL; [1] counts
 * non-positive rho / P, accumulated).  dt is a host scalar here (no device-formed dt).  Limit: Ng <= HYDRO_RTVD_NOALLOC_MAX_GROUPS
 * per call, else HYDRO_E_TOOBIG; other errors as hydro_rtvd_solve_f64 (HYDRO_E_COUNT, _ENUM, _VALUE, _NULL, _ALIGN), > 0 = cudaError_t.
 * No cudaMalloc / cudaFree / allocating library routine is called; the array's device address is looked up once per device
 * (cudaGetSymbolAddress, on the first call with that device current).  ALL calls share the one array, which keeps the last
 * call's contents: nothing in it has to start at zero (every sweep writes what the next sweep reads), but two calls that
 * OVERLAP on the GPU (different streams, or graph branches) RACE on it -- serialise them.  Results equal hydro_rtvd_solve_f64
 * bit for bit (groups are independent; only the number of CTAs differs). */
#define HYDRO_RTVD_NOALLOC_MAX_GROUPS 4096
HYDRO_API int hydro_rtvd_solve_noalloc_f64(const double* in, double* out, double* face_flux, int Ng, double dt, double dh, double gamma,
                                           int order, long long* status, hydro_stream_t stream);

/* Sizes and capabilities. */
HYDRO_API int hydro_min_ghost(int scheme, int recon);                 /* 2/3 (MHM, CTU with PLM/PPM), 3/4 (VL)   */
HYDRO_API int hydro_has_fused(int precision_bytes, int scheme, int recon, int riemann); /* 1 if a fused kernel exists */
/* 1 if that fused kernel's tiles fit in shared memory for ghost width nghost (else AUTO uses the staged path) */
HYDRO_API int hydro_fused_fits(int precision_bytes, int scheme, int recon, int nghost);
/* bytes of opts->workspace that hydro_solve_* may need in HYDRO_IMPL_AUTO mode for any ghost width
 * (0 only when the fused kernel runs for every nghost <= 8) */
HYDRO_API size_t hydro_workspace_bytes(int Ng, int precision_bytes, int scheme, int recon);
/* bytes needed when HYDRO_IMPL_STAGED is forced */
HYDRO_API size_t hydro_staged_workspace_bytes(int Ng, int precision_bytes, int scheme, int recon);
HYDRO_API const char* hydro_strerror(int code);

/* Measurement helper (the FP32 / FP64 ALU peaks the roofline fractions divide by must be MEASURED on
 * the box): launches one register-resident loop of `blocks` x `threads` threads, each running `iters` passes of
 * 8 x 16 independent operations of one kind, on `stream`; the caller times it with CUDA events.
 *   kind 0 FFMA (register operands)   1 FFMA2 (fma.rn.f32x2)   2 DFMA   3 FMUL / FADD alternating
 *        4 FFMA : FMNMX 1:1           5 FFMA2 : FMNMX 1:1      6 MUFU.RSQ   7 FFMA with constant-bank operands
 *        8 / 9: (2 FFMA | 1 FFMA2) + SHF   10 / 11: (6 FFMA | 3 FFMA2) + FSETP + FSEL + SHF   12 / 13: (8 FFMA | 4 FFMA2) +
 *        FSETP + FSEL + MUFU + SHF -- equal arithmetic in scalar and packed form (does FFMA2 relieve the issue port?)
 * scratch: device buffer of >= blocks*threads*8 bytes (never written in practice); *ops_per_launch (host, may be NULL)
 * receives the floating-point operations of the timed kind per launch (FMA = 2; for kinds 4, 5 those of the FMAs only;
 * kind 6: MUFU operations).  Errors: HYDRO_E_ENUM, HYDRO_E_VALUE (threads not a multiple of 32 in [32,512]), HYDRO_E_NULL. */
HYDRO_API int hydro_alu_peak_launch(int kind, int blocks, int threads, int iters, void* scratch, double* ops_per_launch,
                                    hydro_stream_t stream);

#ifdef __cplusplus
}
#endif
#endif /* HYDRO_H_ */
