/* fx.h -- C ABI of libfx.so: the data-parallel hot path of arXiv:1807.01971 (Feltor) on one B200.
 *
 * The preconditioned conjugate-gradient solve of the 2-D discontinuous-Galerkin elliptic equation
 *     div( chi grad phi ) = rho            (the gyro-fluid form div(N grad_perp phi) = n - N is Eq. (1c))
 * built, as the paper prescribes for its "Level 2" algorithms, from "Level 1" vector and matrix primitives only
 * (PAPER.md:75-76): the exactly rounded dot product (section 3.1), axpby and pointwise multiply
 * with a fixed order of explicitly fused operations (section 3.2), and the dG block-stencil
 * matrix-vector product (section 4.1).  "P:n" below = PAPER.md line n; "D:x" = DESIGN.md section x.
 *
 * Conventions for every call
 *   - pointers named *_dev / documented "device" are CUDA device pointers on the current device, owned by the caller,
 *     never retained or freed by the library; pointers documented "host" are ordinary host memory.
 *   - vectors are dense fp64 arrays.  A dG vector of a grid {Nx,Ny,P} has n = P*P*Nx*Ny entries laid out as a
 *     row-major (Ny*P) x (Nx*P) image, x fastest:  idx = ((j*P + l)*Nx + i)*P + k   for cell (i,j), node (k,l)   (D:4).
 *   - every compute call exists in two forms.  NAME_ex(ctx, ...) works on an explicit context (fx_create: one device, one
 *     stream, its own scratch).  The plain NAME(...) uses the default context of the calling thread's current device,
 *     created on first use; its stream is the one set with fx_set_stream (default: the legacy default stream).  Calls are
 *     asynchronous (stream-ordered) except where "synchronises" is stated.
 *   - threads: different contexts are independent (two threads, two streams, two devices may work at the same time).  ONE
 *     context -- in particular the default one -- must be used by one thread at a time, and its stream must not be changed
 *     while work of an earlier call is still in flight (the exact-dot digits and the CG scalars are per-context scratch).
 *   - return value: fx_status.  < 0 is an error (nothing useful was computed), >= 0 is success.  No exceptions,
 *     no aborts.  fx_last_error() returns a thread-local message for the last error.
 *   - there is no CPU fallback: without a CUDA device every compute call returns FX_ECUDA.
 */
#ifndef FX_H
#define FX_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    FX_OK = 0,
    FX_MAXIT = 1,          /* fx_cg_solve: maxit iterations done without meeting tol (not an error)            */
    FX_EINVAL = -1,        /* bad argument (null pointer with n>0, P outside 1..5, overlap where forbidden ...)  */
    FX_ECUDA = -2,         /* CUDA runtime failure; fx_last_error() holds the CUDA string                      */
    FX_ENOMEM = -3,        /* device allocation of library scratch failed                                     */
    FX_EBREAKDOWN = -4     /* fx_cg_solve: p.Sp <= 0 or non-finite (operator not positive definite on p)       */
} fx_status;

/* Boundary kind of one direction.  PER: periodic.  DIR: homogeneous Dirichlet at both walls (the ghost cell is zero).
 * NEU: homogeneous Neumann at both walls (the ghost cell mirrors the interior trace: no jump and no flux correction on
 * the wall face).  DIR_NEU: Dirichlet at the lower wall (x = 0 / y = 0), Neumann at the upper one; needs >= 2 cells in
 * that direction.  NEU_DIR: the reverse.  NEU kinds are for the elliptic operator and the CG solve (a grid without any
 * Dirichlet wall gives a singular operator: constants are its null space); fx_dg_derivative and fx_arakawa take PER
 * and DIR only and return FX_EINVAL otherwise.  (Q23, section 6.9) */
typedef enum { FX_BC_PER = 0, FX_BC_DIR = 1, FX_BC_NEU = 2, FX_BC_DIR_NEU = 3, FX_BC_NEU_DIR = 4 } fx_bc;

/* Grid of Fig. 2 `CartesianGrid2d(x0,x1,y0,y1,P,Nx,Ny)` on the domain [0,lx] x [0,ly]:
 * Nx x Ny cells, P Gauss-Legendre nodes per cell and direction (P = number of polynomial coefficients). */
typedef struct {
    int32_t Nx, Ny, P;     /* Nx,Ny >= 1; 1 <= P <= 5                                                           */
    double lx, ly;         /* > 0                                                                               */
    int32_t bcx, bcy;      /* fx_bc                                                                             */
} fx_grid;

typedef struct {
    int32_t iterations;    /* operator applications inside the loop                                             */
    int32_t status;        /* FX_OK, FX_MAXIT or FX_EBREAKDOWN                                                  */
    double rel_residual;   /* sqrt(r.V.r) / sqrt(b.W.b) at exit                                                  */
} fx_cg_info;

/* ---- contexts ----------------------------------------------------------------------------------
 * The paper's user picks the backend through the vector type (dg::DVec); here the context carries the device
 * and the stream.  fx_create: a context on `device` (a CUDA ordinal) whose work is enqueued on `cuda_stream` (a cudaStream_t
 * passed as void*; NULL = legacy default stream).  It owns its scratch (about 2 KB until a CG solve or a *_host call sizes
 * work vectors) and never retains user pointers.  fx_destroy synchronises the context's stream and frees everything; NULL
 * is ignored.  An _ex call makes the context's device current for its duration and restores the caller's device.       */
typedef struct fx_ctx fx_ctx;
fx_status fx_create(fx_ctx** ctx_out, int32_t device, void* cuda_stream);
void fx_destroy(fx_ctx* ctx);

/* ---- housekeeping ---------------------------------------------------------------------------------------- */

/* Stream (a cudaStream_t passed as void*) used by all later calls of this process; NULL = legacy default.     */
fx_status fx_set_stream(void* cuda_stream);
fx_status fx_set_stream_ex(fx_ctx* ctx, void* cuda_stream);
const char* fx_last_error(void);
/* Release the default contexts of all devices with their scratch (device digits, CG work vectors, events).  Optional; safe
 * to call repeatedly; contexts made by fx_create are not touched.                                               */
void fx_shutdown(void);

/* Test hook for the launch-shape invariance tests (north star: results identical "regardless of grid and block
 * shape").  kernel_id: 0 = exdot, 1 = axpby/pointwise, 2 = dG apply, 3 = fused CG kernels.  grid_dim = number of
 * CTAs (0 = default), block_dim = threads per CTA (0 = default; must be a multiple of 32, <= 1024; the dG apply
 * reads it as warps-per-CTA*32 and grid_dim as rows-per-segment).                                              */
fx_status fx_set_launch(int32_t kernel_id, int32_t grid_dim, int32_t block_dim);
fx_status fx_set_launch_ex(fx_ctx* ctx, int32_t kernel_id, int32_t grid_dim, int32_t block_dim);
/* fx_cg_solve driver: 0 = one kernel per primitive, both dots visit the host; 1 (default) = fused: a single persistent
 * cooperative kernel for grids of up to 2^20 unknowns, two fused kernels per iteration above; 2 = always the two fused
 * kernels; 3 = the persistent kernel whenever possible (< 2^24 unknowns).  Results are bit-identical in every mode.      */
fx_status fx_set_cg_fused(int32_t fused);
fx_status fx_set_cg_fused_ex(fx_ctx* ctx, int32_t fused);
/* Test hook: which dG stencil kernels serve fx_dg_elliptic_apply*, fx_arakawa and fx_cg_solve.  0 (default) = the CTA-tile
 * kernels (2-D TMA staging, D:6.2) whenever the row pitch Nx*P is even and the vectors are 16-byte aligned, else the
 * warp-strip kernels -- except K1 of the two-kernel CG loop, which is the warp-strip kernel for P <= 3 (measured faster)
 * and the tile kernel for P = 4, 5; 1 = always the warp-strip kernels; 2 = the tile kernels wherever they are eligible,
 * K1 included.  Same bits either way.                                                                                    */
fx_status fx_set_dg_path(int32_t path);
fx_status fx_set_dg_path_ex(fx_ctx* ctx, int32_t path);

/* ---- exactly rounded dot product (P:9) ----------------------------------------------------------
 * result = RN( sum_i x[i]*y[i] ), products and sum over the reals, one rounding to nearest-even at the end; the
 * full range of products of doubles is exact (subnormal*subnormal, 2^1000*2^1000 that cancel ...), exact zero
 * gives +0.0, n == 0 gives +0.0; NaN if any input is NaN, any product is 0*inf, or +inf and -inf products both
 * occur; else +-inf if an infinite product occurs or the exact sum rounds beyond DBL_MAX        (D:3.1, Q1-Q6).
 * Bitwise identical for every launch shape.  x, y: device, may alias, n >= 0.                                  */

/* Synchronises; returns the value (NaN and fx_last_error() on failure). */
double fx_exdot(const double* x_dev, const double* y_dev, int64_t n);
/* Context form: result_host (host double; synchronises) and / or result_dev (device double; stream-ordered), at least one. */
fx_status fx_exdot_ex(fx_ctx* ctx, const double* x_dev, const double* y_dev, int64_t n, double* result_host, double* result_dev);
/* Asynchronous form: writes the double to result_dev (device, 8 bytes). */
fx_status fx_exdot_async(const double* x_dev, const double* y_dev, int64_t n, double* result_dev);
fx_status fx_exdot_async_ex(fx_ctx* ctx, const double* x_dev, const double* y_dev, int64_t n, double* result_dev);
/* Allocation-free form, for callers that may not call cudaMalloc (CUDA graph capture, serving loops, harnesses that
 * forbid it): same value, same bits as fx_exdot_async, but no context and no work space -- the long accumulator's device
 * scratch is a file-scope __device__ array of 1728 bytes that every GPU loading the library holds until exit.
 * The call makes no cudaMalloc / cudaFree and calls no allocating routine: a stream-ordered clear of that array and ONE
 * kernel launch on `stream` (a cudaStream_t; NULL = the legacy default stream) of the current device.
 * Limit: 0 <= n <= FX_EXDOT_STATIC_MAX_N (one launch); beyond it FX_EINVAL with a message in fx_last_error().
 * x_dev, y_dev: device, n doubles each, may alias, caller-owned; result_dev: device, 8 bytes, written stream-ordered.
 * The array is shared by every call on that device and keeps the last call's contents (it is cleared before each
 * launch): calls on one stream are ordered and safe; calls that OVERLAP on the GPU (different streams, other host
 * threads' streams) race on it and give undefined values -- use contexts (fx_exdot_async_ex) for concurrency.        */
#define FX_EXDOT_STATIC_MAX_N (1LL << 28)
fx_status fx_exdot_static(const double* x_dev, const double* y_dev, int64_t n, double* result_dev, void* stream);
/* The long accumulator itself: 68 limbs, two's complement, limb k weighs 2^(64k-2176), plus flags
 * {nan, +inf, -inf}.  limbs_host: host uint64[68]; flags_host: host int32[3] or NULL.  Synchronises.          */
fx_status fx_exdot_digits(const double* x_dev, const double* y_dev, int64_t n, uint64_t* limbs_host,
                          int32_t* flags_host, double* result_host);
fx_status fx_exdot_digits_ex(fx_ctx* ctx, const double* x_dev, const double* y_dev, int64_t n, uint64_t* limbs_host,
                             int32_t* flags_host, double* result_host);
/* Host-buffer convenience (the "e2e" path of bench.py): x, y are HOST arrays; copies them to device scratch in
 * chunks on the library stream, accumulates, returns the value.  Synchronises.                                */
double fx_exdot_host(const double* x_host, const double* y_host, int64_t n);
fx_status fx_exdot_host_ex(fx_ctx* ctx, const double* x_host, const double* y_host, int64_t n, double* result_host);

/* Census of the exact reductions' slow paths since the last reset -- the paper's claim under test is that the long
 * accumulator is "rarely invoked".  out_host: host uint64[4] = {elements (product parts) deposited into the long
 * accumulator as exact integers because they reached below the register window, products deposited as 106-bit integer
 * products because TwoProd is not error-free for them (outside [2^-960, 2^1000)), window moves of a warp, 0}; NULL = only
 * reset.  Every reduction kernel of the context counts (dots, sums, the fused CG kernels).  Synchronises.           */
fx_status fx_exdot_stats(uint64_t* out_host, int32_t reset);
fx_status fx_exdot_stats_ex(fx_ctx* ctx, uint64_t* out_host, int32_t reset);

/* Weighted dot sum_i x[i] w[i] y[i] ("the weighted sum ... where w represents for example the volume form") in
 * the reading D:Q14: u = RN(x[i]*w[i]) in fp64, then the exactly rounded dot of u and y.  fx_exsum: the exactly rounded
 * sum of x (EXSUM) = exact dot with ones.  Device pointers, may alias; both synchronise and return the value.      */
double fx_exdot3(const double* x_dev, const double* w_dev, const double* y_dev, int64_t n);
double fx_exsum(const double* x_dev, int64_t n);
fx_status fx_exdot3_ex(fx_ctx* ctx, const double* x_dev, const double* w_dev, const double* y_dev, int64_t n, double* result_host);
fx_status fx_exsum_ex(fx_ctx* ctx, const double* x_dev, int64_t n, double* result_host);
/* binary32 inputs, exact accumulation: RN_double(sum x[i]*y[i]), every product exact.  Synchronises.          */
double fx_exdot_f32(const float* x_dev, const float* y_dev, int64_t n);
fx_status fx_exdot_f32_ex(fx_ctx* ctx, const float* x_dev, const float* y_dev, int64_t n, double* result_host);

/* ---- vector primitives in canonical order (D:3.2) ---------------------------------------------- */

/* y[i] <- fma(alpha, x[i], RN(beta*y[i]));  beta == 0: y[i] <- RN(alpha*x[i]) and y is not read.
 * x, y: device; x may equal y; partial overlap is undefined.                                                   */
fx_status fx_axpby(double alpha, const double* x_dev, double beta, double* y_dev, int64_t n);
fx_status fx_axpby_ex(fx_ctx* ctx, double alpha, const double* x_dev, double beta, double* y_dev, int64_t n);
/* u = RN(alpha*x1[i]); y[i] <- fma(u, x2[i], RN(beta*y[i]));  beta == 0: y[i] <- RN(u*x2[i]), y not read.      */
fx_status fx_pointwise_dot(double alpha, const double* x1_dev, const double* x2_dev, double beta, double* y_dev,
                           int64_t n);
fx_status fx_pointwise_dot_ex(fx_ctx* ctx, double alpha, const double* x1_dev, const double* x2_dev, double beta, double* y_dev,
                              int64_t n);

/* z[i] <- alpha*x1[i]*y1[i] + beta*x2[i]*y2[i] + gamma*z[i], the fused product the paper adds "to raise the work per call"
 * (P:414).  Canonical order (D:Q22): a = RN(alpha*x1); b = RN(beta*x2); t = gamma == 0 ? RN(b*y2) : fma(b, y2, RN(gamma*z));
 * z = fma(a, y1, t).  gamma == 0: z is not read.  Inputs may alias each other and z.                                     */
fx_status fx_pointwise_dot2(double alpha, const double* x1_dev, const double* y1_dev, double beta, const double* x2_dev,
                            const double* y2_dev, double gamma, double* z_dev, int64_t n);
fx_status fx_pointwise_dot2_ex(fx_ctx* ctx, double alpha, const double* x1_dev, const double* y1_dev, double beta, const double* x2_dev,
                               const double* y2_dev, double gamma, double* z_dev, int64_t n);

/* ---- dG elliptic operator (construction D:3.3, operation order D:3.4) -------------------------
 * S = Fx^T diag(W chi) Fx + Fy^T diag(W chi) Fy + (jump terms), symmetric; A = diag(V) S ~ -div(chi grad .),
 * V = 1/W the inverse dG weights.  chi, x, y: device vectors of the grid; y must not overlap x or chi.         */
fx_status fx_dg_elliptic_apply(const fx_grid* grid, const double* chi_dev, const double* x_dev, double* y_dev);     /* y = A x */
fx_status fx_dg_elliptic_apply_sym(const fx_grid* grid, const double* chi_dev, const double* x_dev, double* y_dev); /* y = S x */
fx_status fx_dg_elliptic_apply_ex(fx_ctx* ctx, const fx_grid* grid, const double* chi_dev, const double* x_dev, double* y_dev);
fx_status fx_dg_elliptic_apply_sym_ex(fx_ctx* ctx, const fx_grid* grid, const double* chi_dev, const double* x_dev, double* y_dev);
/* dG weights W ("volume" of Fig. 2) and V = 1/W; either pointer may be NULL.  Device vectors.           */
fx_status fx_dg_weights(const fx_grid* grid, double* w_dev, double* v_dev);
fx_status fx_dg_weights_ex(fx_ctx* ctx, const fx_grid* grid, double* w_dev, double* v_dev);
/* The reference-element tables the kernels use, for the cross-check against the oracle's own tables.
 * out_host: host double[5*P + 4*P*P] = xi,w,L,R,B (P each) then T0,T0L,WW,D (P*P each, row-major).  No GPU.   */
fx_status fx_dg_tables(int32_t P, double* out_host);

/* ---- 3-D product grids (D:Q24) -----------------------------------------------------------------------------
 * The paper's applications are "2D/3D drift-/gyro-fluid simulations" with derivatives "on product spaces";
 * its elliptic equation is the perpendicular one, div(chi grad_perp phi) = rho (Eq. 1c).  Reading D:Q24: Nz planes
 * of the 2-D grid with one node per plane in z (cell height hz = lz/Nz).  A vector stores plane after plane
 * (idx3 = plane * P*P*Nx*Ny + idx2); the operator acts in every plane, the planes meet in the dot products of CG.  Weights (the
 * volume form): W3 = RN(hz * W2), V3 = RN(1/W3).  sym != 0: y = S3 x = RN(hz * (S2 x_plane)); sym == 0: y = A3 x = A2 x_plane.   */
typedef struct {
    int32_t Nx, Ny, Nz, P;
    double lx, ly, lz;
    int32_t bcx, bcy;      /* fx_bc of the x and y directions (z carries no derivative) */
} fx_grid3;
fx_status fx_dg3_elliptic_apply(const fx_grid3* grid, const double* chi_dev, const double* x_dev, double* y_dev, int32_t sym);
fx_status fx_dg3_elliptic_apply_ex(fx_ctx* ctx, const fx_grid3* grid, const double* chi_dev, const double* x_dev, double* y_dev, int32_t sym);
fx_status fx_dg3_weights(const fx_grid3* grid, double* w_dev, double* v_dev);
fx_status fx_dg3_weights_ex(fx_ctx* ctx, const fx_grid3* grid, double* w_dev, double* v_dev);
/* fx_cg_solve on the product grid: one system over all planes (S3 phi = W3 o (-rho), preconditioner V3, global exact dots).  */
fx_status fx_cg3_solve(const fx_grid3* grid, const double* chi_dev, const double* rho_dev, double* phi_dev,
                       double tol, int32_t maxit, fx_cg_info* info);
fx_status fx_cg3_solve_ex(fx_ctx* ctx, const fx_grid3* grid, const double* chi_dev, const double* rho_dev, double* phi_dev,
                          double tol, int32_t maxit, fx_cg_info* info);

/* ---- stand-alone dG derivatives: the paper's "dxdy" primitive (P:240, P:321 / Table 3; D:6.7, Q21) -----------------
 * y <- alpha * M x + beta * y (beta == 0: y is not read), M = d/dx (direction 0) or d/dy (direction 1) of the grid with its
 * boundary condition in that direction; flux 0 = forward (the F of the elliptic operator), 1 = backward (-W^-1 F^T W),
 * 2 = centred (their mean); 3 = the un-normed jump matrix of that direction (sum over the faces of [v][u]: block row n has
 * diagonal R R^T + L L^T and off-diagonals -R L^T, -L R^T; no 1/h), the third matrix of the paper's primitive "for dx, dy and
 * jump".  x, y: device vectors of the grid; y must not overlap x.                                                        */
fx_status fx_dg_derivative(const fx_grid* grid, int32_t direction, int32_t flux, double alpha, const double* x_dev, double beta,
                           double* y_dev);
fx_status fx_dg_derivative_ex(fx_ctx* ctx, const fx_grid* grid, int32_t direction, int32_t flux, double alpha, const double* x_dev,
                              double beta, double* y_dev);
/* Arakawa bracket out = {f, g} = f_x g_y - f_y g_x in Arakawa's conserving form with centred dG derivatives (the
 * second composite the paper benchmarks, Fig. 6a), defined as the nine calls of D:6.8: 4 derivatives, 3 fused pointwise
 * products, 2 accumulating derivatives (the three products run in one kernel, with the bits of the three calls).
 * f, g, out: device vectors of the grid; out must not overlap f or g.  Six work vectors are kept by the library.        */
fx_status fx_arakawa(const fx_grid* grid, const double* f_dev, const double* g_dev, double* out_dev);
fx_status fx_arakawa_ex(fx_ctx* ctx, const fx_grid* grid, const double* f_dev, const double* g_dev, double* out_dev);
/* The derivative tables for the cross-check against the oracle: host double[2*P*P + 2*P] = TT interior, TT first
 * Dirichlet cell (P*P each, row-major), cN, cP.  No GPU.                                                               */
fx_status fx_dg_dtables(int32_t P, int32_t flux, double* out_host);

/* ---- preconditioned CG (algorithm D:3.5) ------------------------------------------------------
 * Solves div(chi grad phi) = rho as S phi = W o (-rho) with preconditioner V; every dot product exactly rounded;
 * stops when sqrt(r.V.r) <= tol*sqrt(b.W.b) (tested after every iteration) or after maxit iterations.
 * chi, rho: device (read only); phi: device, in = phi0, out = phi; info: host or NULL.  Synchronises.
 * Returns info->status.                                                                                       */
fx_status fx_cg_solve(const fx_grid* grid, const double* chi_dev, const double* rho_dev, double* phi_dev,
                      double tol, int32_t maxit, fx_cg_info* info);
fx_status fx_cg_solve_ex(fx_ctx* ctx, const fx_grid* grid, const double* chi_dev, const double* rho_dev, double* phi_dev,
                         double tol, int32_t maxit, fx_cg_info* info);
/* Host-buffer convenience (bench.py "e2e"): chi, rho, phi are HOST arrays of the grid's n doubles.            */
fx_status fx_cg_solve_host(const fx_grid* grid, const double* chi_host, const double* rho_host, double* phi_host,
                           double tol, int32_t maxit, fx_cg_info* info);
fx_status fx_cg_solve_host_ex(fx_ctx* ctx, const fx_grid* grid, const double* chi_host, const double* rho_host, double* phi_host,
                              double tol, int32_t maxit, fx_cg_info* info);

/* Timing hook for bench.py: with enable != 0, fx_cg_solve (fused driver) records CUDA events on its stream around
 * the kernels of every enable-th iteration of the loop (1 = every iteration; the events between the kernels cost
 * about 9 us per sampled iteration on a B200, so bench.py samples every 8th) and around the whole loop.
 * fx_cg_last_profile then returns, for the most recent solve: the device time of the whole loop, the device time of each
 * of the two kernels K1 (direction update + apply + dot) and K2 (updates + preconditioner + dot) summed over the sampled
 * iterations and scaled to the loop's iteration count, and that count.  ms_host: host double[4] = {loop, K1, K2, 0}.  */
fx_status fx_cg_profile(int32_t enable);
fx_status fx_cg_last_profile(double* ms_host, int32_t* iterations_host);
fx_status fx_cg_profile_ex(fx_ctx* ctx, int32_t enable);
fx_status fx_cg_last_profile_ex(fx_ctx* ctx, double* ms_host, int32_t* iterations_host);

/* Timing hook for the latency-bandwidth sweep (the paper reports average run times of back-to-back calls):
 * launches one primitive `reps` times (after one untimed call) between two CUDA events on the library stream and
 * returns the average milliseconds per call in *ms_host.  kind: 0 = exdot(a,b) result left on the device,
 * 1 = axpby(0.7,a,-0.3,c), 2 = pointwise_dot(1,a,b,0,c), 3 = dG apply_sym(grid; chi=a, x=b, y=c), 4 = dG apply (normed),
 * 5 = exdot(a,b) returned to the host every call (the paper's GPU dot latency), 6 = axpby(0.7,a,1,c),
 * 7 = weighted dot(a,b,c) device-resident, 8 = exact sum(a) device-resident; with a grid: 9/10 = d/dx, d/dy forward,
 * 11/12 = d/dx, d/dy centred, each as c <- 0.7 M a - 0.3 c; 13 = Arakawa bracket c = {a, b} (nine calls);
 * 14 = the fp64 issue roof: a kernel of (SM count * 8) CTAs x 256 threads x 8 independent chains x 4096 dependent fused
 * multiply-adds and no memory traffic (the second roof of the exact dot and the stencil; a, b unused).
 * a, b, c: device vectors of n doubles (kinds 3,4,9-13: n must equal the grid's size).  Synchronises.               */
fx_status fx_time_primitive(int32_t kind, const fx_grid* grid, const double* a_dev, const double* b_dev, double* c_dev,
                            int64_t n, int32_t reps, double* ms_host);
fx_status fx_time_primitive_ex(fx_ctx* ctx, int32_t kind, const fx_grid* grid, const double* a_dev, const double* b_dev, double* c_dev,
                               int64_t n, int32_t reps, double* ms_host);

/* Number of kernels this library has launched since load, over all contexts (bench.py's "gpu_launches").      */
int64_t fx_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* FX_H */
