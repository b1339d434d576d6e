/* include/gamer_hydro.h — C ABI of the B200-native GAMER hydro hot path (arXiv 1007.3818).
 *
 * What the library computes. PAPER.md:15 (§2): "a new GPU hydrodynamic solver based on the MUSCL-Hancock
 * method. This approach contains four steps, namely, the spatial data reconstruction, the half-step
 * prediction, the Riemann solver, and the full-step update. We apply the unsplit finite volume method for
 * the three-dimensional evolution, and the Roe's solver is adopted for the Riemann problem."
 * PAPER.md:27 (§2): "it requires only a five-point stencil in each spatial direction" (=> 2 ghost cells) and
 * "the operation of preparing the ghost-zone data is conducted by CPU": the caller hands over a batch of
 * patch groups WITH their ghost shells already filled; one call advances every group by one time step.
 * The numerical details the paper leaves open are fixed in DESIGN.md §3 (readings R1–R21).
 *
 * All functions: extern "C", never throw, never exit; return 0 on success or a GAMER_HYDRO_* code.
 * Concurrency: the library serves ONE device per process (the first one it is used on; a second device returns
 * GAMER_HYDRO_INVALID_ARG: run one process per GPU). gamer_hydro_step / _f64, gamer_hydro_max_speed,
 * gamer_hydro_fill_ghosts, gamer_hydro_step_grid and gamer_hydro_advance may be called concurrently from several
 * host threads on different streams: gamer_hydro_max_speed and gamer_hydro_advance LEASE a reduction slot of their own
 * for as long as they run (an advance: for all its steps) — 64 leases at a time, the 65th concurrent call returns
 * GAMER_HYDRO_BUSY rather than share one — and calls that need the library's one scratch buffer (the shape-generic
 * kernels) are chained by an event, i.e. they run one after the other; growing that buffer, reading its address and
 * enqueueing on it happen under one lock. Process-global and NOT thread-safe: gamer_hydro_set_path,
 * gamer_hydro_set_guard_map, gamer_hydro_status (test / diagnostic plumbing), gamer_hydro_step_host (it owns the
 * library's three internal streams) and gamer_hydro_advance on the DUO path (it ping-pongs with one library-owned
 * array).
 * Pointers are DEVICE pointers unless the name says host. Nothing here takes or returns a torch type.
 *
 * Layouts (x fastest, then y, then z; `real` = float or double):
 *   U_in            real[n_groups][5][S][S][S],  S = N + 2*ghost; variables (rho, mx, my, mz, E);
 *                   interior cell (i,j,k) sits at (i+ghost, j+ghost, k+ghost). Only the innermost two ghost
 *                   layers are read; of those, corner ghosts and layer-2 edge ghosts are never read.
 *   U_out           real[n_groups][5][N][N][N]
 *   boundary_fluxes real[n_groups][6][5][N][N] or NULL (skipped). Faces ordered -x,+x,-y,+y,-z,+z (face index
 *                   -1/2 and N-1/2 along the axis); in-face index [k][j] for x faces, [k][i] for y faces,
 *                   [j][i] for z faces. Each entry is the Roe flux DENSITY ALONG THE +AXIS (not the outward
 *                   normal) of (rho, mx, my, mz, E), exactly the value used in the update.
 * Ownership: the caller owns every buffer; the library never allocates, frees or keeps them. U_in is
 * read-only; outputs must not alias U_in. Device pointers must be 16-byte aligned.
 * Equation of state: ideal gas, E = P/(gamma-1) + rho |v|^2 / 2.  limiter: 0 = MinMod, 1 = van Leer, 2 = MC.
 */
#ifndef GAMER_HYDRO_H
#define GAMER_HYDRO_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct CUstream_st* cudaStream_t;

enum {
  GAMER_HYDRO_OK = 0,
  GAMER_HYDRO_INVALID_ARG = 1, /* null U_in/U_out, n_groups<0, N<1, ghost<2, dt/dx not finite or <=0, gamma<=1,
                                  unknown limiter, misaligned pointer */
  GAMER_HYDRO_UNSUPPORTED = 2, /* shape the library has no kernel for */
  GAMER_HYDRO_CUDA_ERROR = 3,  /* a CUDA call failed; gamer_hydro_strerror(3) carries the CUDA message */
  GAMER_HYDRO_NOT_SM100 = 4,   /* the device is not compute capability 10.x */
  GAMER_HYDRO_TOO_LARGE = 5,   /* gamer_hydro_max_speed_noalloc: more patch groups than its fixed scratch array holds */
  GAMER_HYDRO_BUSY = 6         /* gamer_hydro_max_speed / gamer_hydro_advance: 64 such calls are already in flight */
};

enum { GAMER_HYDRO_MINMOD = 0, GAMER_HYDRO_VANLEER = 1, GAMER_HYDRO_MC = 2 /* monotonized central, R3b */ };

/* Riemann-solver flags of gamer_hydro_step_ex (PAPER.md:15 names only "the Roe's solver", which
 * is flags = 0): Harten & Hyman's entropy fix of the acoustic waves; Einfeldt's HLLE flux wherever an intermediate
 * state of Roe's linearisation is non-physical. Readings R8b / R8c of DESIGN.md §14. */
enum { GAMER_HYDRO_FLAG_ENTROPY_FIX = 1, GAMER_HYDRO_FLAG_HLLE_FALLBACK = 2 };

/* kernel selection for gamer_hydro_set_path: AUTO picks FUSED when N == 16, else GENERIC. FUSED is the
 * performance path (fp32: one column per thread, the two lanes of every packed f32x2 instruction carry two
 * consecutive z planes; fp64: one cell per thread, scalar). FUSED_SCALAR forces the scalar fused kernel in
 * fp32 as well and FUSED_DUO the one-cell-per-thread kernel whose packed lanes carry two directions (the
 * kernel the fused-halo step of gamer_hydro_step_grid is built on): structurally different implementations
 * of the same step (tests, comparisons). */
enum {
  GAMER_HYDRO_PATH_AUTO = 0,
  GAMER_HYDRO_PATH_GENERIC = 1,
  GAMER_HYDRO_PATH_FUSED = 2,
  GAMER_HYDRO_PATH_FUSED_SCALAR = 3,
  GAMER_HYDRO_PATH_FUSED_DUO = 4
};

/* One-time, idempotent, process-global set-up for `device`: checks the compute capability, raises the
 * dynamic shared-memory limits of the kernels, allocates the device status block and (for the generic
 * path and the host-buffer path) scratch sized for min(max_groups, internal chunk) groups of N^3 cells
 * with `bytes_per_real` (4 or 8). Synchronous. gamer_hydro_step* call it with defaults when it was not
 * called. Calling it again with larger sizes grows the scratch. */
int gamer_hydro_alloc(int max_groups, int N, int ghost, int bytes_per_real, int device);

/* Releases everything gamer_hydro_alloc created (synchronises the device first). */
void gamer_hydro_free(void);

/* One MUSCL-Hancock + Roe time step on n_groups patch groups, fp32. Enqueues on `stream` and
 * returns without synchronising; re-entrant across streams. Deterministic: each cell's arithmetic sequence
 * is fixed, so results do not depend on n_groups or on the launch geometry. n_groups == 0 is a no-op.
 * Non-positive rho or P in the input is the caller's fault: no hang, garbage confined to that group.
 * This is the signature fixed by BASELINE.json:north_star. */
int gamer_hydro_step(const float* U_in_with_ghosts, float* U_out, float* boundary_fluxes, int n_groups, int N,
                     int ghost, float dt, float dx, float gamma, int limiter, cudaStream_t stream);

/* Same step in fp64 (parity target 1e-11 against the fp64 oracle). */
int gamer_hydro_step_f64(const double* U_in_with_ghosts, double* U_out, double* boundary_fluxes, int n_groups,
                         int N, int ghost, double dt, double dx, double gamma, int limiter, cudaStream_t stream);

/* The step with the robustness variants of SURVEY.md §8(f) rank 4: `flags` = GAMER_HYDRO_FLAG_* bits,
 * and midplane_fluxes (DEVICE, may be NULL) = real[n_groups][3][5][N][N], the Roe fluxes on the three MID-planes of each
 * group (the faces at index N/2 - 1/2 along x, y, z — the internal patch boundaries of a group of 2 x 2 x 2 patches, which
 * the AMR flux fix-up needs beside the outer faces), each in the in-face layout of the outer faces of the same axis; N
 * must be even. With flags = 0 and midplane_fluxes = NULL this is gamer_hydro_step (same kernels, same bits); otherwise
 * the step runs in the scalar fused kernel (N = 16) or the shape-generic kernels. Other arguments, errors and
 * execution semantics as gamer_hydro_step. */
int gamer_hydro_step_ex(const float* U_in_with_ghosts, float* U_out, float* boundary_fluxes, float* midplane_fluxes,
                        int n_groups, int N, int ghost, float dt, float dx, float gamma, int limiter, int flags,
                        cudaStream_t stream);
int gamer_hydro_step_ex_f64(const double* U_in_with_ghosts, double* U_out, double* boundary_fluxes,
                            double* midplane_fluxes, int n_groups, int N, int ghost, double dt, double dx, double gamma,
                            int limiter, int flags, cudaStream_t stream);

/* Same fp32 step with HOST buffers (pinned memory recommended; pageable works but serialises the copies).
 * The batch is streamed through the device in chunks: H2D copy, kernel and D2H copy of consecutive chunks
 * overlap on internal streams — the B200 counterpart of the paper's overlap of data transfer with
 * computation ("concurrent execution between CPU and GPU"). Synchronous: returns
 * when U_out / boundary_fluxes (host) are complete. chunk_groups <= 0 picks the default. */
int gamer_hydro_step_host(const float* h_U_in_with_ghosts, float* h_U_out, float* h_boundary_fluxes, int n_groups,
                          int N, int ghost, float dt, float dx, float gamma, int limiter, int chunk_groups);

/* ---- the steps either side of the hot path, for device-resident multi-step runs on ONE uniform grid of
 * gx x gy x gz patch groups (group index x-fastest: g = (bz * gy + by) * gx + bx). The paper does both on the CPU
 * ("the operation of preparing the ghost-zone data is conducted by CPU"); here they are plain
 * streaming kernels so that a run never leaves the GPU. bytes_per_real is 4 or 8. ---- */

/* CFL signal speed (reading R15): *h_max (HOST) = max over the interior cells of all groups of
 * |vx| + |vy| + |vz| + 3 c_s, c_s = sqrt(gamma max(P, 0) / rho). U is a DEVICE array [n_groups][5][S][S][S],
 * S = N + 2 ghost (ghost = 0 for a U_out array). Synchronises `stream`. */
int gamer_hydro_max_speed(const void* U, int bytes_per_real, int n_groups, int N, int ghost, double gamma,
                          double* h_max, cudaStream_t stream);

/* The CFL signal speed of gamer_hydro_max_speed (reading R15, fp32) for callers that cannot afford a device
 * allocation, now or later in the run. Two kinds of caller are meant. An AMR code that fills the GPU with its patch
 * pools at start-up: a cudaMalloc made on its behalf in the middle of a run can fail for lack of memory, hours in. And
 * a time loop that keeps copies and kernels of several streams in flight ("concurrent execution between CPU
 * and GPU"): cudaMalloc and cudaFree wait for the whole device, so one allocation stalls every stream. The other
 * entry points allocate on first use (gamer_hydro_alloc: status block, scratch, staging buffers). This one calls no
 * cudaMalloc, no cudaFree and no library routine that allocates, and does not run gamer_hydro_alloc: its only working
 * memory is one fixed array inside the library image, 256.25 KiB (a 256-byte header and one word per patch group),
 * which every GPU that loads the library holds until the process exits.
 *   U       float[n_groups][5][S][S][S], S = N + 2*ghost (ghost = 0 for a U_out array), DEVICE, read-only
 *   d_max   one float, DEVICE, 4-byte aligned, owned by the caller: receives the maximum over the interior cells of all
 *           groups of |vx| + |vy| + |vz| + 3 c_s; NaN if any cell is NaN (same rule and same arithmetic as
 *           gamer_hydro_max_speed, which returns the value to the host instead)
 * Enqueues a 4-byte clear of the array's counter and one kernel on `stream` and returns without synchronising; read
 * *d_max on the same stream (for instance with cudaMemcpyAsync into pinned memory) when it is needed.
 * Limits and rules:
 *   - 1 <= n_groups <= gamer_hydro_max_speed_noalloc_limit() (65536); more returns GAMER_HYDRO_TOO_LARGE and enqueues
 *     nothing. Split a larger batch and take the maximum of the parts.
 *   - Call it with the device that owns U, d_max and `stream` current. The first call on each device looks up where that
 *     device keeps its copy of the array (cudaGetSymbolAddress) and checks the compute capability; make that first call
 *     before any stream capture begins. Later calls only enqueue.
 *   - All calls on one device share the array, and it keeps the last call's contents. The counter that must start at
 *     zero is cleared by every call itself. Two calls whose kernels can overlap on the GPU (different streams with no
 *     event between them) race on the array and both results are then undefined: order them with an event, or keep
 *     them on one stream, where they run one after the other.
 * Errors: GAMER_HYDRO_INVALID_ARG (null or misaligned pointer, n_groups < 1, N < 1, ghost < 0, gamma <= 1),
 * GAMER_HYDRO_TOO_LARGE, GAMER_HYDRO_NOT_SM100, GAMER_HYDRO_UNSUPPORTED (device ordinal >= 64), GAMER_HYDRO_CUDA_ERROR. */
int gamer_hydro_max_speed_noalloc(const float* U, int n_groups, int N, int ghost, float gamma, float* d_max,
                                  cudaStream_t stream);

/* Largest n_groups gamer_hydro_max_speed_noalloc accepts (65536: twice the headline batch of 32768 groups). */
int gamer_hydro_max_speed_noalloc_limit(void);

/* Same-level ghost-shell refill (reading R16): rebuilds every stored cell of U_in_with_ghosts
 * [G][5][S][S][S] — interior and ghost shell — from the interior arrays U_out [G][5][N][N][N] of the groups that
 * own the cells; per axis bc = 0 wraps periodically, bc = 1 copies the nearest interior cell (outflow). Device
 * pointers, enqueue-and-return; the two arrays must not alias. */
int gamer_hydro_fill_ghosts(const void* U_out, void* U_in_with_ghosts, int bytes_per_real, int gx, int gy, int gz, int N,
                            int ghost, int bc_x, int bc_y, int bc_z, cudaStream_t stream);

/* One fp32 step of a FULLY PERIODIC uniform grid with the halo exchange fused into the step kernel: besides U_out
 * and boundary_fluxes (as gamer_hydro_step) the kernel writes every updated cell straight into
 * U_next_with_ghosts [G][5][20][20][20] — its own interior position and the ghost shells of the up to seven
 * neighbouring groups it borders — so that U_next is the complete ghosted input of the next step (bit-identical to
 * gamer_hydro_fill_ghosts applied to U_out), and accumulates the signal-speed maximum of the new state for
 * gamer_hydro_advance. N = 16, ghost = 2 only (else GAMER_HYDRO_UNSUPPORTED); U_next must not alias U. */
int gamer_hydro_step_grid(const float* U_with_ghosts, float* U_out, float* boundary_fluxes, float* U_next_with_ghosts,
                          int gx, int gy, int gz, int N, int ghost, float dt, float dx, float gamma, int limiter,
                          cudaStream_t stream);

/* n_steps time steps of the fp32 path on one uniform grid without leaving the device: per step
 * dt = float(cfl * dx / max signal speed) (fp64 on the host from the device-side maximum, R15/R11), then
 * gamer_hydro_step, then the ghost refill of gamer_hydro_fill_ghosts (whose kernel also accumulates the next maximum). U (ghost shells filled on entry) holds the final state with
 * refilled ghost shells on return, U_out the interiors of the last step, boundary_fluxes (may be NULL) those of
 * the last step; h_dts (HOST, n_steps floats, may be NULL) receives the time steps taken. One 4-byte
 * device-to-host read and one stream synchronisation per step. With GAMER_HYDRO_PATH_FUSED_DUO selected, a fully
 * periodic grid of 16^3 groups uses gamer_hydro_step_grid instead of step + refill, ping-ponging between U and a
 * second ghosted array the library allocates (and keeps). A state without a finite positive signal speed ends the
 * loop with GAMER_HYDRO_INVALID_ARG: a NaN cell makes the device maximum NaN, and so does a cell with rho <= 0 as long as
 * its pressure expression stays positive (the sound speed is then the root of a negative number). NOT caught: a cell with
 * rho > 0 and P <= 0 enters with c_s = 0 (R15's max(P, 0)), and a cell with rho < 0 whose clamped pressure is 0 drops out
 * of the maximum; the loop then continues on that state with the time step of the other cells — such cells are counted,
 * never repaired (gamer_hydro_status, R10). On every return, error or not, U holds the state after the steps completed
 * so far. */
int gamer_hydro_advance(float* U_with_ghosts, float* U_out, float* boundary_fluxes, int gx, int gy, int gz, int N,
                        int ghost, int bc_x, int bc_y, int bc_z, int n_steps, float cfl, float dx, float gamma,
                        int limiter, float* h_dts, cudaStream_t stream);

/* ---- second workload: the relaxing-TVD solver. PAPER.md:13 (§2): "the second-order relaxing
 * total variation diminishing (TVD) method (Trac & Pen 2003)", dimensionally split; it needs "seven points"
 * per direction, i.e. THREE ghost cells. One call = one time step of every group: three 1-D sweeps with the full dt, in
 * the order x, y, z (sweep = 0) or z, y, x (sweep = 1; callers alternate). Each sweep: half step with the first-order
 * upwind fluxes of the relaxed system (freezing speed |v| + c_s per cell), full step with van-Leer-limited second-order
 * fluxes on the half-step state (readings RT1–RT8). fp32.
 *   U_in_with_ghosts  float[n_groups][5][S][S][S], S = N + 2*ghost, DEVICE, 16-byte aligned, read-only
 *   U_out             float[n_groups][5][N][N][N], DEVICE, must not alias U_in
 * N = 16 and ghost = 3 only (GAMER_HYDRO_UNSUPPORTED otherwise); no boundary fluxes (RT7). Enqueues on `stream` and
 * returns; re-entrant across streams; deterministic. Errors as gamer_hydro_step. */
int gamer_rtvd_step(const float* U_in_with_ghosts, float* U_out, int n_groups, int N, int ghost, float dt, float dx,
                    float gamma, int sweep, cudaStream_t stream);

/* Diagnostics accumulated since the last call (and reset by it): number of cells whose predicted face
 * states failed the positivity guard and fell back to first order (R7), and number of updated
 * cells with rho <= 0 or P <= 0 (R10: counted, never floored). Synchronises the device. Either pointer may
 * be NULL. */
int gamer_hydro_status(unsigned long long* guard_cells, unsigned long long* nonpositive_out);

/* Debug aid of the parity harness (R7: cells where GPU and oracle DISAGREE on the guard are excluded from
 * the parity maximum). With device_map != NULL every later step call marks the cells whose predicted states fell
 * back to first order: device_map[g][k+1][j+1][i+1] = 1, unsigned char [n_groups][N+2][N+2][N+2] in DEVICE memory,
 * owned and zeroed by the caller, indices -1 .. N per axis (first ghost layer included). NULL (the default) switches
 * it off. Process-global, synchronises the device; the map is written on the rare fallback path only. The group index
 * g is the one of the step call's own batch: do not combine the map with gamer_hydro_step_host, which steps the batch
 * in chunks (every chunk would mark the map from g = 0 again). */
int gamer_hydro_set_guard_map(unsigned char* device_map);

/* The same aid for the HLLE fallback of gamer_hydro_step_ex (GAMER_HYDRO_FLAG_HLLE_FALLBACK is a discontinuous switch:
 * a face whose intermediate state is marginal can take the other branch in fp32 than in the fp64 oracle). With
 * device_map != NULL every later step_ex call marks the faces that took the HLLE branch:
 * device_map[g][axis][k][j][i] = 1, unsigned char [n_groups][3][N+1][N+1][N+1] in DEVICE memory, owned and zeroed by the
 * caller; the face is the one on the lower side of cell (i, j, k) along the axis (index N = the upper outer face).
 * NULL (the default) switches it off. Process-global, synchronises the device; same caveat about
 * gamer_hydro_step_host as the guard map. */
int gamer_hydro_set_hlle_map(unsigned char* device_map);

/* Forces a kernel path (tests, benchmarking); GAMER_HYDRO_PATH_AUTO restores the default. */
int gamer_hydro_set_path(int path);

/* Number of kernel launches the library has enqueued since it was loaded (bench.py's gpu_launches). */
unsigned long long gamer_hydro_launch_count(void);

/* Static string for a return code; for GAMER_HYDRO_CUDA_ERROR the last CUDA error message. */
const char* gamer_hydro_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* GAMER_HYDRO_H */
