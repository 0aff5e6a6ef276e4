/* =====================================================================================
 * mhd.h -- C ABI of the B200 patch-group MHD solver (libmhd.so).
 *
 * The hot path of GAMER-MHD (Zhang, Schive & Chiueh 2018; citations are PAPER.md:<line>):
 * the unsplit second-order Godunov update of a batch of ghost-zoned patch groups
 * by the VL / MUSCL-Hancock scheme (7 steps) or the CTU
 * scheme (8 steps), with PLM/PPM reconstruction, an HLLE/HLLD/Roe Riemann
 * solver and constrained transport of the face-centred magnetic field
 * (Eq. 13), plus the CFL time-step reduction.
 * Where the paper is silent the readings R1-R18 of DESIGN.md apply.
 *
 * Every step runs in hand-written CUDA kernels for sm_100a.  There is no CPU fallback: every
 * call fails with MHD_ECUDA when no CUDA device is usable.
 *
 * ---- array layouts (per group, contiguous; groups outermost; SoA; index order [k][j][i], x fastest) ----
 * N = ps2 interior cells per side, g = nghost, T = N + 2g.  Real = float (MHD_FP32) or double (MHD_FP64).
 *   U_in  [G][5][T][T][T]      (rho, Mx, My, Mz, e); e includes 1/2 Bc^2, Bc = mean of the two faces (Eq. 5)
 *   B_in  [G]{ Bx[T][T][T+1] | By[T][T+1][T] | Bz[T+1][T][T] }   Bx[k][j][i] = field on face i-1/2 of cell (i,j,k) (Fig. 1)
 *   U_out [G][5][N][N][N]
 *   B_out [G]{ Bx[N][N][N+1] | By[N][N+1][N] | Bz[N+1][N][N] }   interior faces incl. both boundary planes
 *   flux_out [G][9][5][N][N]   plane p = 3*d + s; d = normal (x,y,z); s = 0 lower boundary face plane (face index 0),
 *                              1 mid plane (index N/2, boundary between the two patches), 2 upper boundary (index N);
 *                              5 = time-centred fluxes of (rho,Mx,My,Mz,e) used in the final update, NOT multiplied
 *                              by dt or area; [N][N] = (t2,t1) transverse cell indices, t1 fastest, (d,t1,t2) cyclic
 *   emf_out  [G][9][2][(N+1)*N] same 9 planes; component 0 = E_t1 on the plane's edges along t1, [N+1 in t2][N in t1];
 *                              component 1 = E_t2 on edges along t2, [N in t2][N+1 in t1]
 * ===================================================================================== */
#ifndef MHD_B200_H
#define MHD_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mhd_solver mhd_solver; /* opaque; owns the device workspace, streams and staging buffers */

typedef enum { MHD_FP32 = 0, MHD_FP64 = 1 } mhd_precision;
typedef enum { MHD_VL = 0, MHD_CTU = 1 } mhd_scheme;            /* PAPER.md:191-197 / :176-183 */
typedef enum { MHD_PLM = 0, MHD_PPM = 1 } mhd_recon;
typedef enum { MHD_HLLE = 0, MHD_HLLD = 1, MHD_ROE = 2 } mhd_riemann;
typedef enum { MHD_LIM_PRIM = 0, MHD_LIM_CHAR = 1 } mhd_limvar; /* limiter in primitive / characteristic variables */
typedef enum { MHD_LIMITER_MC = 0, MHD_LIMITER_MINMOD = 1, MHD_LIMITER_VANLEER = 2 } mhd_limiter; /* slope limiter; the paper
                                              names none: MC is the default reading (R5), the others NEXT-4 variants */

typedef struct {
  int ps2;          /* N: interior cells per side of a patch group; 16 = 2 patches of 8; even, 8..64 */
  int nghost;       /* g: >= 3 for PLM, >= 4 for PPM (R8); exactly the ghost width of the arrays passed in */
  double gamma;     /* ratio of specific heats, > 1 (5/3 in every paper test) */
  int scheme;       /* mhd_scheme */
  int recon;        /* mhd_recon */
  int riemann;      /* mhd_riemann */
  int limvar;       /* mhd_limvar */
  int prec;         /* mhd_precision: element type of every array argument */
  double min_dens;  /* floors applied to DERIVED primitive states only (R9); conserved output is never floored */
  double min_pres;
  double emf_tie;   /* CT upwinding tie (R10a): a face mass flux m with |m| dt/dh <= emf_tie * (mean density of the
                       two cells) counts as zero and takes the centred average; <= 0 selects 1e-12 (FP64) / 1e-5 (FP32) */
  int max_groups;   /* largest ngroups of one mhd_advance call (bounds nothing but argument checking) */
  int device;       /* CUDA device ordinal */
  int limiter;      /* mhd_limiter (0 = MC) */
  int hcorr;        /* NEXT-4 variant, 0 / 1: H-correction of the Roe solver (R19: every dissipation speed of the corrector
                       pass raised to eta^H, the largest fast-characteristic jump over the face and the 8 transverse faces of its two
                       cells).  Needs riemann = MHD_ROE and nghost one larger than the scheme alone (4 with PLM, 5 with PPM), else
                       MHD_EINVAL.  Every scheme: VL / CTU with PLM / PPM */
} mhd_config;

/* MHD_ESTATE: a call that returns a time step (mhd_dt_reduce, mhd_advance_dt, mhd_advance_host_dt, mhd_grid_dt,
 * mhd_grid_advance_dt) found no finite positive signal speed -- the state holds NaN or infinite values (a cell with a NaN
 * input reports an infinite speed, so the maximum cannot drop it).  The arrays have been written; *dt_out is not usable. */
enum { MHD_OK = 0, MHD_EINVAL = -1, MHD_ECUDA = -2, MHD_ENOMEM = -3, MHD_ESTATE = -4, MHD_ELIMIT = -5 };
/* MHD_ELIMIT: the call needs more than the fixed capacity of a no-allocation entry point (mhd_dt_reduce_noalloc). */

/* Create a solver.  Allocates the device workspace (for min(max_groups, what fits a 6 GB budget) groups: larger
 * batches are processed in equal slices).  Returns MHD_EINVAL for a bad configuration (incl. too small a ghost width), MHD_ECUDA /
 * MHD_ENOMEM for device errors.  *out is NULL on failure. */
int mhd_create(const mhd_config* cfg, mhd_solver** out);
int mhd_destroy(mhd_solver* s);

/* Element counts PER GROUP of the six arrays (any pointer may be NULL). */
int mhd_sizes(const mhd_solver* s, size_t* n_U_in, size_t* n_B_in, size_t* n_U_out, size_t* n_B_out,
              size_t* n_flux, size_t* n_emf);

/* Advance ngroups patch groups by dt with cell size dh (one pass of the whole scheme, PAPER.md:176-183 / :191-197).
 * All array pointers are DEVICE pointers owned by the caller, laid out as above in the solver's precision.
 * flux_out and emf_out may each be NULL.  Asynchronous on cuda_stream (a cudaStream_t; NULL = default stream);
 * allocates nothing and never synchronises.  Outputs must not alias inputs.  ngroups = 0 is a no-op.
 * Errors: MHD_EINVAL (null pointer, ngroups < 0 or > max_groups, dt or dh not finite/positive), MHD_ECUDA (launch). */
int mhd_advance(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out,
                void* flux_out, void* emf_out, int ngroups, double dt, double dh, void* cuda_stream);

/* Same update with HOST pointers (pinned memory gives the overlap; pageable memory works but serialises).
 * The batch is cut into chunks of chunk_groups; chunk c runs H2D -> kernels -> D2H on stream c % nstreams so that
 * copy-in, compute and copy-out of successive chunks overlap.  Blocking.  1 <= nstreams <= 8,
 * 1 <= chunk_groups <= max_groups.  flux_out / emf_out may be NULL. */
int mhd_advance_host(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out,
                     void* flux_out, void* emf_out, int ngroups, double dt, double dh,
                     int chunk_groups, int nstreams);

/* mhd_advance_host with the CFL reduction of the new state fused into every chunk's final update (see mhd_advance_dt):
 * the complete path S0-S9 through HOST buffers.  dt_out (required) and maxspeed_out (nullable) are HOST pointers; outputs
 * bit-identical to mhd_advance_host, dt bit-identical to mhd_advance_dt.  ngroups >= 1.  Blocking. */
int mhd_advance_host_dt(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out,
                        void* flux_out, void* emf_out, int ngroups, double dt, double dh,
                        int chunk_groups, int nstreams, double cfl, double* dt_out, double* maxspeed_out);

/* CFL time step (R13): dt = cfl * dh / max over interior cells and directions d of
 * (|v_d| + c_f,d), cell-centred B = face mean.  U, B: DEVICE arrays of ngroups groups whose ghost width is
 * nghost_of_arrays (0: the U_out/B_out layout; cfg.nghost: the U_in/B_in layout).  dt_out (required) and
 * maxspeed_out (nullable) are HOST pointers; the call synchronises cuda_stream. */
int mhd_dt_reduce(mhd_solver* s, const void* U, const void* B, int ngroups, int nghost_of_arrays,
                  double dh, double cfl, double* dt_out, double* maxspeed_out, void* cuda_stream);

/* mhd_advance followed by mhd_dt_reduce(U_out, B_out, ngroups, 0, dh, cfl, ...) as ONE call: the full update (S8,
 * PAPER.md:183, :197) also evaluates the CFL speed (S9) of every cell it writes and reduces it on the
 * device, so the new state is not read back for the time step.  Arguments as mhd_advance (DEVICE pointers) plus cfl;
 * dt_out (required) and maxspeed_out (nullable) are HOST pointers.  Results (outputs, dt, maxspeed) are bit-identical
 * to the two separate calls.  ngroups >= 1.  Blocking: synchronises cuda_stream like mhd_dt_reduce. */
int mhd_advance_dt(mhd_solver* s, const void* U_in, const void* B_in, void* U_out, void* B_out, void* flux_out,
                   void* emf_out, int ngroups, double dt, double dh, double cfl, double* dt_out, double* maxspeed_out,
                   void* cuda_stream);

/* mhd_dt_reduce for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same CFL reduction (R13) with NO solver object, no cudaMalloc / cudaFree / allocating
 * library call, and no host synchronisation.  The scratch memory of the reduction (one partial maximum per 256-cell block and an
 * arrival counter) is a fixed array of the library's device image: (MHD_NOALLOC_MAX_BLOCKS + 32) * 8 bytes = 513 KB, held on
 * every GPU that loads the library until the process exits.  It runs on the CURRENT device.
 *   prec: MHD_FP32 / MHD_FP64, the element type of U and B (DEVICE arrays, layouts of mhd_dt_reduce: ps2 interior cells per
 *   side, nghost_of_arrays ghost cells in the arrays, 0 ... 8); gamma, min_dens, min_pres as in mhd_config (no defaults here).
 *   dt_speed_out: DEVICE pointer to two doubles, written by the kernel: [0] = dt = cfl * dh / maxspeed, [1] = maxspeed -- the bits
 *   that mhd_dt_reduce returns for the same arguments.  A state with NaN / infinite values gives maxspeed = +inf and dt = 0 (the
 *   call is asynchronous and cannot return MHD_ESTATE): the caller checks.
 * Limit: ngroups * ceil(ps2^3 / 256) <= MHD_NOALLOC_MAX_BLOCKS and ngroups <= 65535 (4096 groups of 16^3), else MHD_ELIMIT and
 * nothing is launched.  Asynchronous on cuda_stream: one memset node (the counter) and one kernel, both capturable.  The first call
 * on a device asks the driver for the array's address (cudaGetSymbolAddress): make it outside a capture.
 * All calls share the one array: calls that overlap on the GPU (other streams, concurrently replayed graphs) race -- serialise. */
#define MHD_NOALLOC_MAX_BLOCKS 65536
int mhd_dt_reduce_noalloc(int prec, const void* U, const void* B, int ngroups, int ps2, int nghost_of_arrays, double gamma,
                          double min_dens, double min_pres, double dh, double cfl, double* dt_speed_out, void* cuda_stream);

/* Cumulative event counters since creation (density floors, pressure floors, Roe->HLLE fallbacks).
 * Synchronises the device; asynchronous kernel faults surface here as MHD_ECUDA. */
int mhd_get_stats(mhd_solver* s, unsigned long long* n_floor_dens, unsigned long long* n_floor_pres,
                  unsigned long long* n_riemann_fallback);

/* Number of kernel launches issued by this solver since creation (bench.py's gpu_launches). */
unsigned long long mhd_launch_count(const mhd_solver* s);

/* ---- device-side preparation and closing steps for a uniform PERIODIC grid ----
 * Grid arrays (DEVICE pointers, solver precision, x fastest): U[5][nz][ny][nx], bx[nz][ny][nx+1], by[nz][ny+1][nx],
 * bz[nz+1][ny][nx]; the last face of each direction duplicates the first.  nx, ny, nz are multiples of ps2 and >= nghost;
 * the grid is cut into (nx/ps2)(ny/ps2)(nz/ps2) <= max_groups patch groups, group index (gz*my + gy)*mx + gx.
 * mhd_grid_pack fills U_in / B_in (layouts of mhd_advance) with periodic ghost zones; mhd_grid_unpack stores U_out / B_out
 * back (every cell owns its three lower faces; the duplicate last faces are rewritten).  mhd_grid_advance = pack ->
 * mhd_advance -> unpack in place on the grid through solver-owned staging buffers (allocated on first use; asynchronous
 * on cuda_stream afterwards).  mhd_grid_dt is mhd_dt_reduce on the grid layout (synchronises cuda_stream). */
int mhd_grid_pack(mhd_solver* s, const void* U, const void* bx, const void* by, const void* bz, int nx, int ny, int nz,
                  void* U_in, void* B_in, void* cuda_stream);
int mhd_grid_unpack(mhd_solver* s, const void* U_out, const void* B_out, int nx, int ny, int nz, void* U, void* bx, void* by,
                    void* bz, void* cuda_stream);
int mhd_grid_advance(mhd_solver* s, void* U, void* bx, void* by, void* bz, int nx, int ny, int nz, double dt, double dh,
                     void* cuda_stream);
/* mhd_grid_advance followed by mhd_grid_dt of the new grid state as one call (the final update reduces the CFL speed,
 * see mhd_advance_dt): the time step of the next step costs no extra pass over the grid.  dt_out (required) and
 * maxspeed_out (nullable) are HOST pointers; bit-identical to the two separate calls; synchronises cuda_stream. */
int mhd_grid_advance_dt(mhd_solver* s, void* U, void* bx, void* by, void* bz, int nx, int ny, int nz, double dt, double dh,
                        double cfl, double* dt_out, double* maxspeed_out, void* cuda_stream);
int mhd_grid_dt(mhd_solver* s, const void* U, const void* bx, const void* by, const void* bz, int nx, int ny, int nz, double dh,
                double cfl, double* dt_out, double* maxspeed_out, void* cuda_stream);

/* ---- the AMR correction operation on a static two-level mesh ----
 * Coarse level: a periodic grid in the layout of mhd_grid_* (DEVICE pointers) cut into patch groups in grid order; fine
 * level: the patch groups (cell size dh_c / 2) covering ONE refined box of coarse cells lo[d] .. hi[d]-1, ordered z
 * outermost, x fastest.  lo, hi: HOST int[3], multiples of ps2/2, ps2/2 <= lo < hi <= n - ps2/2.
 * mhd_amr_restrict: coarse cells of the box <- volume average of 8 fine cells (U_out of the fine groups), coarse faces of
 * the box including its surface <- area average of 4 fine faces (B_out).
 * mhd_amr_fixup: every leaf coarse cell sharing a face with the box gets  U += -/+ (dt/dh_c) (w_f <F_fine> - w_c F_coarse)
 * (upper / lower face of the cell), <F_fine> the mean of the 4 fine fluxes of that face; every leaf coarse face touching an
 * edge of the box surface gets the Eq. 13 update of the jump  w_f <E_fine> - w_c E_coarse  of that edge.  flux_c / emf_c:
 * flux_out / emf_out of ALL coarse groups of the step being corrected; flux_f / emf_f: those of the fine groups.  With
 * both levels advanced by the same dt, w_c = w_f = 1; with sub-cycling call once per fine step with w_f = 1/nsub and
 * w_c = 1 on the first call, 0 afterwards.  Call the fix-up BEFORE the restriction is irrelevant: they touch disjoint data.
 * Asynchronous on cuda_stream.  MHD_EINVAL for a misaligned box. */
int mhd_amr_restrict(mhd_solver* s, const void* U_f, const void* B_f, const int* lo, const int* hi, void* Uc, void* bxc,
                     void* byc, void* bzc, int nx, int ny, int nz, void* cuda_stream);
int mhd_amr_fixup(mhd_solver* s, const void* flux_c, const void* emf_c, const void* flux_f, const void* emf_f, const int* lo,
                  const int* hi, double dt, double dh_c, double w_c, double w_f, void* Uc, void* bxc, void* byc, void* bzc,
                  int nx, int ny, int nz, void* cuda_stream);

/* ---- creating new fine grids ----
 * Coarse level: a periodic grid in the layout of mhd_grid_* (DEVICE pointers, solver precision).  The box of coarse cells
 * lo[d] .. hi[d]-1 (HOST int[3], 0 <= lo < hi <= n) is refined by 2: U_f[5][2nbz][2nby][2nbx] <- conservative
 * piecewise-linear interpolation with MC-limited slopes (the mean of the 8 fine cells is the coarse cell); bx_f[2nbz][2nby]
 * [2nbx+1], by_f[2nbz][2nby+1][2nbx], bz_f[2nbz+1][2nby][2nbx] <- Balsara (2001) divergence-free interpolation: fine faces
 * on a coarse face from the MC-limited linear profile of that face (their mean is the coarse value), interior fine faces
 * from the polynomial of Eq. 17 carried to 3-D (21 coefficients fixed by the interface and divergence conditions,
 * PAPER.md:213-219), so that the fine field is divergence-free to round-off when the coarse one is.  Coarse neighbours
 * are periodic; every coarse face of the box is interpolated (no copy from pre-existing fine neighbours: the box is
 * taken to be surrounded by coarse cells).  nb[d] = hi[d] - lo[d].  Asynchronous on cuda_stream.  MHD_EINVAL for a bad box. */
int mhd_amr_prolong(mhd_solver* s, const void* Uc, const void* bxc, const void* byc, const void* bzc, int nx, int ny, int nz,
                    const int* lo, const int* hi, void* U_f, void* bx_f, void* by_f, void* bz_f, void* cuda_stream);

/* Per-stage device timing for the roofline report: when on, every stage launch is bracketed by CUDA events on its
 * stream (up to 16384 launches since the last mhd_set_profiling call; later ones are not recorded).
 * mhd_get_profile synchronises the device, fills the summed milliseconds and launch counts of each stage
 * (arrays of at least 16 entries) and returns the number of stages; mhd_profile_stage_name names stage i. */
int mhd_set_profiling(mhd_solver* s, int on);
int mhd_get_profile(mhd_solver* s, double* ms_per_stage, unsigned long long* launches_per_stage, int nstages);
const char* mhd_profile_stage_name(int stage);

/* Register-only FMA-chain micro-kernel: measured FP32 (prec=0) or FP64 (prec=1) FMA peak of this device in
 * TFLOP/s (2 flop per FMA), used as the ALU roofline denominator beside the nominal figure. */
int mhd_measure_fma_peak(int device, int prec, double* tflops_out);

/* Message for a return code; for MHD_ECUDA the last CUDA error string seen by this thread. */
const char* mhd_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* MHD_B200_H */
