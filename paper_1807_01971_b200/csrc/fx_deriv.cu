// fx_deriv.cu -- stand-alone dG derivatives  y <- alpha * M x + beta * y  (the paper's "dxdy" primitive: derivatives in x and
// y on product spaces; m = 3 memory passes, P:321 / Table 3).  SURVEY 8f-2; definition DESIGN.md 6.7 / Q21.
//
// Canonical order per line, cell n, node k (the test oracle restates it independently):
//     a = chain_m(TT[k][m], u_{n,m});  a = fma(cP[k], tR_{n-1}, a);  a = fma(cN[k], tL_{n+1}, a);  d = RN((2/h) * a)
//     y = beta == 0 ? RN(alpha * d) : fma(alpha, d, RN(beta * y))
// The paper stores the few distinct P x P blocks once so that the matrix costs no memory traffic and makes P
// a template parameter; here the blocks are kernel parameters (constant bank), and the two directions get the
// thread mapping that suits the x-fastest layout:
//   * d/dx: a lane owns one cell of one image row (P contiguous doubles), neighbour traces by warp shuffle, strips of 30
//     cells with a one-cell halo on each side (as the elliptic apply);
//   * d/dy: a lane owns one image COLUMN and marches through the cells of a row segment -- every load and store is a
//     fully coalesced 256-byte row, the previous cell's top trace is carried in a register, the next cell's values are
//     loaded one step ahead and become the current cell.
// HBM roofline: 24 B per unknown (16 B for beta == 0), ~P + 8 fp64 operations.

#include <string.h>

#include "fx_internal.h"
#include "fx_dgb.cuh"

struct DdParams {
    int Nx, Ny, bc, beta0;
    int rows_per_seg, nseg, nstrip;
    double s, alpha, beta;
    double TT[2][FX_PMAX][FX_PMAX], cN[FX_PMAX], cP[FX_PMAX], L[FX_PMAX], R[FX_PMAX];
};

#define DD_CHAIN(acc, COEF, VAL)                         \
    {                                                    \
        acc = __dmul_rn(COEF(0), VAL(0));                \
        _Pragma("unroll") for (int m_ = 1; m_ < P; ++m_) \
            acc = __fma_rn(COEF(m_), VAL(m_), acc);      \
    }

template <int P>
__device__ __forceinline__ double dd_out(const DdParams& g, int k, bool first, const double (&u)[P], double tRp, double tLn) {
    double a;
#define CT(m) (first ? g.TT[1][k][m] : g.TT[0][k][m])
#define UU(m) u[m]
    DD_CHAIN(a, CT, UU)
#undef CT
    a = __fma_rn(g.cP[k], tRp, a);
    a = __fma_rn(g.cN[k], tLn, a);
    return __dmul_rn(g.s, a);
}

__device__ __forceinline__ double dd_axpby(const DdParams& g, double d, double yold) {
    return g.beta0 ? __dmul_rn(g.alpha, d) : __fma_rn(g.alpha, d, __dmul_rn(g.beta, yold));
}

// ---- d/dx: warp = strip of 30 cells x rows_per_seg image rows ----------------------------------------------------------
template <int P>
__global__ void __launch_bounds__(256) k_dg_dx(const __grid_constant__ DdParams g, const double* __restrict__ x, double* __restrict__ y) {
    const int wpb = blockDim.x >> 5, lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * wpb + (threadIdx.x >> 5);
    if (w >= (long long)g.nstrip * g.nseg) return;
    const int seg = (int)(w / g.nstrip), strip = (int)(w % g.nstrip);
    const int rows = g.Ny * P, Nx = g.Nx;
    const long long pitch = (long long)Nx * P;
    const int r0 = seg * g.rows_per_seg;
    int r1 = r0 + g.rows_per_seg;
    if (r1 > rows) r1 = rows;
    const int ci = strip * FX_STRIP - 1 + lane;
    const bool outside = ci < 0 || ci >= Nx, dir = g.bc == 1;
    int cw = ci;
    if (outside) { cw = ci % Nx; if (cw < 0) cw += Nx; }
    const bool ghost = outside && (dir || ci < -1 || ci > Nx);
    const bool produce = lane >= 1 && lane <= FX_STRIP && ci < Nx;
    const bool first = dir && ci == 0;
    for (int r = r0; r < r1; ++r) {
        const double* q = x + (long long)r * pitch + (long long)cw * P;
        double u[P], yo[P];
#pragma unroll
        for (int k = 0; k < P; ++k) u[k] = __ldg(q + k);
        double* yq = y + (long long)r * pitch + (long long)cw * P;
        if (!g.beta0 && produce) {
#pragma unroll
            for (int k = 0; k < P; ++k) yo[k] = yq[k];
        }
        double tL, tR;
#define CL(m) g.L[m]
#define CR(m) g.R[m]
        DD_CHAIN(tL, CL, UU)
        DD_CHAIN(tR, CR, UU)
        if (ghost) { tL = 0.0; tR = 0.0; }
        const double tLn = __shfl_down_sync(0xffffffffu, tL, 1), tRp = __shfl_up_sync(0xffffffffu, tR, 1);
        if (produce) {
#pragma unroll
            for (int k = 0; k < P; ++k) yq[k] = dd_axpby(g, dd_out<P>(g, k, first, u, tRp, tLn), g.beta0 ? 0.0 : yo[k]);
        }
    }
}

// ---- d/dy: lane = image column, warp marches through the cells [j0, j1) of its row segment -------------------------------
template <int P>
__global__ void __launch_bounds__(256) k_dg_dy(const __grid_constant__ DdParams g, const double* __restrict__ x, double* __restrict__ y) {
    const int wpb = blockDim.x >> 5, lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * wpb + (threadIdx.x >> 5);
    if (w >= (long long)g.nstrip * g.nseg) return;
    const int seg = (int)(w / g.nstrip), strip = (int)(w % g.nstrip);      // strip = block of 32 columns
    const long long pitch = (long long)g.Nx * P;
    const long long col = (long long)strip * 32 + lane;
    if (col >= pitch) return;                                             // no warp-collective operations below
    const int Ny = g.Ny;
    const bool dir = g.bc == 1;
    const int j0 = seg * g.rows_per_seg;
    int j1 = j0 + g.rows_per_seg;
    if (j1 > Ny) j1 = Ny;
    double uc[P], un[P], u2[P], tRp;
    const double* xc = x + col;
#pragma unroll
    for (int l = 0; l < P; ++l) uc[l] = __ldg(xc + ((long long)j0 * P + l) * pitch);
    {
        const int jn0 = (j0 + 1 == Ny) ? 0 : j0 + 1;
#pragma unroll
        for (int l = 0; l < P; ++l) un[l] = __ldg(xc + ((long long)jn0 * P + l) * pitch);
    }
    if (j0 == 0 && dir) tRp = 0.0;
    else {
        const int jp = j0 == 0 ? Ny - 1 : j0 - 1;
        double up[P];
#pragma unroll
        for (int l = 0; l < P; ++l) up[l] = __ldg(xc + ((long long)jp * P + l) * pitch);
#define UP(m) up[m]
        DD_CHAIN(tRp, CR, UP)
#undef UP
    }
    for (int j = j0; j < j1; ++j) {
        const bool ghost = dir && j + 1 == Ny;                           // un holds row 0 then; its trace is forced to zero
        if (j + 1 < j1) {                                                // two cells ahead: in flight while this cell is computed
            int j2 = j + 2; if (j2 >= Ny) j2 -= Ny;
#pragma unroll
            for (int l = 0; l < P; ++l) u2[l] = __ldg(xc + ((long long)j2 * P + l) * pitch);
        }
        double yo[P];
        double* yc = y + col + (long long)j * P * pitch;
        if (!g.beta0) {
#pragma unroll
            for (int l = 0; l < P; ++l) yo[l] = yc[l * pitch];
        }
        double tLn, tR;
#define UN(m) un[m]
#define UC(m) uc[m]
        DD_CHAIN(tLn, CL, UN)
        if (ghost) tLn = 0.0;
        DD_CHAIN(tR, CR, UC)
        const bool first = dir && j == 0;
#pragma unroll
        for (int l = 0; l < P; ++l) yc[l * pitch] = dd_axpby(g, dd_out<P>(g, l, first, uc, tRp, tLn), g.beta0 ? 0.0 : yo[l]);
        tRp = tR;
#pragma unroll
        for (int l = 0; l < P; ++l) { uc[l] = un[l]; un[l] = u2[l]; }
    }
}
#undef UN
#undef UC
#undef UU
#undef CL
#undef CR

fx_status fx_launch_derivative(FxCtx* c, const fx_grid* g, int dir, int flux, double alpha, const double* x, double beta, double* y) {
    fx_tables t;
    fx_dtables d;
    if (fx_make_tables(g->P, &t) != 0 || fx_make_dtables(g->P, flux, &d) != 0) { fx_set_error("fx_dg_derivative: bad P or flux"); return FX_EINVAL; }
    DdParams p;
    memset(&p, 0, sizeof(p));
    const int P = g->P;
    p.Nx = g->Nx; p.Ny = g->Ny; p.bc = dir == 0 ? g->bcx : g->bcy; p.beta0 = beta == 0.0;
    volatile double h = dir == 0 ? g->lx / g->Nx : g->ly / g->Ny;
    p.s = flux == 3 ? 1.0 : 2.0 / h; p.alpha = alpha; p.beta = beta;      // (the jump matrix carries no 1/h)
    for (int k = 0; k < P; ++k) {
        p.cN[k] = d.cN[k]; p.cP[k] = d.cP[k]; p.L[k] = t.L[k]; p.R[k] = t.R[k];
        for (int m = 0; m < P; ++m) { p.TT[0][k][m] = d.TT[0][k][m]; p.TT[1][k][m] = d.TT[1][k][m]; }
    }
    const long long target = (long long)c->num_sms * 64;               // warps wanted (light kernels: ~2 waves of 32 per SM)
    const int wpb = 8;
    if (dir == 0) {
        p.nstrip = (g->Nx + FX_STRIP - 1) / FX_STRIP;
        const int rows = g->Ny * P;
        long long nseg = target / p.nstrip; if (nseg < 1) nseg = 1;
        int rps = (int)((rows + nseg - 1) / nseg); if (rps < 1) rps = 1;
        if (c->launch[2][0] > 0) rps = c->launch[2][0];
        if (rps > rows) rps = rows;
        p.rows_per_seg = rps; p.nseg = (rows + rps - 1) / rps;
    } else {
        p.nstrip = (int)(((long long)g->Nx * P + 31) / 32);
        long long nseg = target / p.nstrip; if (nseg < 1) nseg = 1;
        int rps = (int)((g->Ny + nseg - 1) / nseg); if (rps < 4) rps = 4;   // each segment re-reads one cell row
        if (c->launch[2][0] > 0) rps = c->launch[2][0];
        if (rps > g->Ny) rps = g->Ny;
        p.rows_per_seg = rps; p.nseg = (g->Ny + rps - 1) / rps;
    }
    const long long warps = (long long)p.nstrip * p.nseg;
    const int grid = (int)((warps + wpb - 1) / wpb);
#define FX_DD_LAUNCH(K)                                                         \
    switch (P) {                                                                \
    case 1: K<1><<<grid, wpb * 32, 0, c->stream>>>(p, x, y); break;             \
    case 2: K<2><<<grid, wpb * 32, 0, c->stream>>>(p, x, y); break;             \
    case 3: K<3><<<grid, wpb * 32, 0, c->stream>>>(p, x, y); break;             \
    case 4: K<4><<<grid, wpb * 32, 0, c->stream>>>(p, x, y); break;             \
    default: K<5><<<grid, wpb * 32, 0, c->stream>>>(p, x, y); break;            \
    }
    if (dir == 0) { FX_DD_LAUNCH(k_dg_dx) } else { FX_DD_LAUNCH(k_dg_dy) }
    c->launches++;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

extern "C" fx_status fx_dg_derivative_ex(fx_ctx* c, const fx_grid* g, int32_t direction, int32_t flux, double alpha, const double* x, double beta,
                                      double* y) {
    FX_ENTER(c, "fx_dg_derivative");
    if (!fx_grid_ok(g) || !fx_grid_deriv_ok(g) || !x || !y || direction < 0 || direction > 1 || flux < 0 || flux > 3) {
        fx_set_error("fx_dg_derivative: bad grid, direction, flux or null pointer"); return FX_EINVAL;
    }
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P;
    if (x < y + n && y < x + n) { fx_set_error("fx_dg_derivative: y overlaps x"); return FX_EINVAL; }
    return fx_launch_derivative(c, g, direction, flux, alpha, x, beta, y);
}
extern "C" fx_status fx_dg_derivative(const fx_grid* g, int32_t direction, int32_t flux, double alpha, const double* x, double beta,
                                      double* y) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_dg_derivative_ex(c, g, direction, flux, alpha, x, beta, y) : FX_ECUDA;
}

extern "C" fx_status fx_dg_dtables(int32_t P, int32_t flux, double* out) {
    fx_dtables d;
    if (!out || fx_make_dtables(P, flux, &d) != 0) { fx_set_error("fx_dg_dtables: bad arguments"); return FX_EINVAL; }
    double* o = out;
    for (int v = 0; v < 2; ++v) for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = d.TT[v][k][m];
    for (int k = 0; k < P; ++k) *o++ = d.cN[k];
    for (int k = 0; k < P; ++k) *o++ = d.cP[k];
    return FX_OK;
}

// ---- Arakawa bracket as the paper runs it: nine calls of the primitives --------------------------------
// The three fused products of the bracket in one pass (6 vectors in, 3 out instead of 3 x (4 in, 1 out)); per element the
// operation sequence of three fx_pointwise_dot2 calls with alpha = 1/3, beta = -1/3, gamma = 0:
//   out = 1/3 (fx gy - fy gx),  h1 = 1/3 (f gy - g fy),  h2 = 1/3 (g fx - f gx)
__global__ void __launch_bounds__(512) k_arakawa_products(double a, double b, const double* __restrict__ f, const double* __restrict__ g,
                                                          const double* __restrict__ fx, const double* __restrict__ fy,
                                                          const double* __restrict__ gx, const double* __restrict__ gy,
                                                          double* __restrict__ out, double* __restrict__ h1, double* __restrict__ h2, long long n) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double F = f[i], G = g[i], FX = fx[i], FY = fy[i], GX = gx[i], GY = gy[i];
        out[i] = __fma_rn(__dmul_rn(a, FX), GY, __dmul_rn(__dmul_rn(b, FY), GX));
        h1[i] = __fma_rn(__dmul_rn(a, F), GY, __dmul_rn(__dmul_rn(b, G), FY));
        h2[i] = __fma_rn(__dmul_rn(a, G), FX, __dmul_rn(__dmul_rn(b, F), GX));
    }
}

// ---- the bracket in two kernels on the CTA-tile stencil (fx_dgb.cuh) ------------------------------------------------------
#define DGB_NS(STAGE) ((STAGE) == 0 ? 4 : 3)
template <int P, int STAGE>
__global__ void __launch_bounds__(DgtCfg<P>::NT)
k_arakawa_tile(const __grid_constant__ DbParams g, const __grid_constant__ DgtTile t, const __grid_constant__ CUtensorMap m0,
               const __grid_constant__ CUtensorMap m0h, const __grid_constant__ CUtensorMap m1, const __grid_constant__ CUtensorMap m1h,
               const __grid_constant__ CUtensorMap m2, const __grid_constant__ CUtensorMap m2h, double* __restrict__ o0,
               double* __restrict__ o1, double* __restrict__ o2) {
    __shared__ __align__(8) unsigned long long bars[DGB_NS(STAGE)];
    if (threadIdx.x == 0) {
        for (int s = 0; s < DGB_NS(STAGE); ++s) fx_mbar_init(fx_smem_addr(bars) + 8u * s, 1u);
        fx_mbar_fence_init();
        fx_tma_prefetch_desc(&m0); fx_tma_prefetch_desc(&m1);
    }
    __syncthreads();
    const CUtensorMap* const mm[3] = {&m0, &m1, &m2};
    const CUtensorMap* const mh[3] = {&m0h, &m1h, &m2h};
    dgb_tile<P, DgtCfg<P>::NBX, DGB_NS(STAGE), STAGE>(g, t, mm, mh, o0, o1, o2, bars, (int)(blockIdx.x % t.ntx), (int)(blockIdx.x / t.ntx));
}

template <int P>
static fx_status launch_arakawa_tile(FxCtx* c, const fx_grid* g, const double* f, const double* gg, double* out, double* h1, double* h2) {
    constexpr int NBX = DgtCfg<P>::NBX;
    typedef DgtGeom<P, NBX, 2, DGB_NS(0)> GA;
    typedef DgtGeom<P, NBX, 3, DGB_NS(1)> GB;
    fx_tables t;
    fx_dtables d;
    if (fx_make_tables(P, &t) != 0 || fx_make_dtables(P, 2, &d) != 0) { fx_set_error("fx_arakawa: tables"); return FX_EINVAL; }
    DbParams p;
    memset(&p, 0, sizeof(p));
    p.Nx = g->Nx; p.Ny = g->Ny; p.bcx = g->bcx; p.bcy = g->bcy;
    volatile double hx = g->lx / g->Nx, hy = g->ly / g->Ny;
    p.sx = 2.0 / hx; p.sy = 2.0 / hy; p.third = 1.0 / 3.0;
    for (int k = 0; k < P; ++k) {
        p.cN[k] = d.cN[k]; p.cP[k] = d.cP[k]; p.L[k] = t.L[k]; p.R[k] = t.R[k];
        for (int m = 0; m < P; ++m) { p.TT[0][k][m] = d.TT[0][k][m]; p.TT[1][k][m] = d.TT[1][k][m]; }
    }
    const int pitch = g->Nx * P, rows = g->Ny * P;
    CUtensorMap mf, mfh, mg, mgh, m1, m1h, m2, m2h, mo, moh;
    fx_status s;
    if ((s = fx_dgt_make_map(&mf, f, pitch, rows, GA::BW, P)) != FX_OK || (s = fx_dgt_make_map(&mfh, f, pitch, rows, GA::HW, P)) != FX_OK ||
        (s = fx_dgt_make_map(&mg, gg, pitch, rows, GA::BW, P)) != FX_OK || (s = fx_dgt_make_map(&mgh, gg, pitch, rows, GA::HW, P)) != FX_OK ||
        (s = fx_dgt_make_map(&m1, h1, pitch, rows, GB::BW, P)) != FX_OK || (s = fx_dgt_make_map(&m1h, h1, pitch, rows, GB::HW, P)) != FX_OK ||
        (s = fx_dgt_make_map(&m2, h2, pitch, rows, GB::BW, P)) != FX_OK || (s = fx_dgt_make_map(&m2h, h2, pitch, rows, GB::HW, P)) != FX_OK ||
        (s = fx_dgt_make_map(&mo, out, pitch, rows, GB::BW, P)) != FX_OK || (s = fx_dgt_make_map(&moh, out, pitch, rows, GB::HW, P)) != FX_OK)
        return s;
    DgtTile ta, tb;
    const int occa = fx_func_occ(c, (const void*)k_arakawa_tile<P, 0>, GA::NT, GA::SMEM, true);
    const int occb = fx_func_occ(c, (const void*)k_arakawa_tile<P, 1>, GB::NT, GB::SMEM, true);
    fx_dgt_shape(c, g, NBX, c->num_sms * occa, &ta);
    fx_dgt_shape(c, g, NBX, c->num_sms * occb, &tb);
    k_arakawa_tile<P, 0><<<ta.ntx * ta.nseg, GA::NT, GA::SMEM, c->stream>>>(p, ta, mf, mfh, mg, mgh, mg, mgh, out, h1, h2);
    k_arakawa_tile<P, 1><<<tb.ntx * tb.nseg, GB::NT, GB::SMEM, c->stream>>>(p, tb, m1, m1h, m2, m2h, mo, moh, out, nullptr, nullptr);
    c->launches += 2;
    FX_CUDA(cudaGetLastError());
    return FX_OK;
}

extern "C" fx_status fx_arakawa_ex(fx_ctx* c, const fx_grid* g, const double* f, const double* gg, double* out) {
    FX_ENTER(c, "fx_arakawa");
    if (!fx_grid_ok(g) || !fx_grid_deriv_ok(g) || !f || !gg || !out) { fx_set_error("fx_arakawa: bad grid (PER / DIR only) or null pointer"); return FX_EINVAL; }
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P;
    if ((f < out + n && out < f + n) || (gg < out + n && out < gg + n)) { fx_set_error("fx_arakawa: out overlaps an input"); return FX_EINVAL; }
    if (c->ara_cap < n) {
        if (c->ara_vec) { cudaStreamSynchronize(c->stream); cudaFree(c->ara_vec); c->ara_vec = nullptr; c->ara_cap = 0; }
        if (cudaMalloc(&c->ara_vec, (size_t)6 * n * sizeof(double)) != cudaSuccess) {
            fx_set_error("Arakawa work space: %s", cudaGetErrorString(cudaGetLastError())); return FX_ENOMEM;
        }
        c->ara_cap = n;
    }
    double *fx_ = c->ara_vec, *fy_ = fx_ + n, *gx_ = fy_ + n, *gy_ = gx_ + n, *h1 = gy_ + n, *h2 = h1 + n;
    // two kernels on the tile stencil (9 vector passes) where TMA's rules allow; else the seven launches below (23 passes)
    if (c->dg_path != 1 && fx_dgt_eligible(g, f, gg, out)) {
        switch (g->P) {
        case 1: return launch_arakawa_tile<1>(c, g, f, gg, out, h1, h2);
        case 2: return launch_arakawa_tile<2>(c, g, f, gg, out, h1, h2);
        case 3: return launch_arakawa_tile<3>(c, g, f, gg, out, h1, h2);
        case 4: return launch_arakawa_tile<4>(c, g, f, gg, out, h1, h2);
        default: return launch_arakawa_tile<5>(c, g, f, gg, out, h1, h2);
        }
    }
    const double third = 1.0 / 3.0;
    fx_status s;
    if ((s = fx_launch_derivative(c, g, 0, 2, 1.0, f, 0.0, fx_)) != FX_OK) return s;
    if ((s = fx_launch_derivative(c, g, 1, 2, 1.0, f, 0.0, fy_)) != FX_OK) return s;
    if ((s = fx_launch_derivative(c, g, 0, 2, 1.0, gg, 0.0, gx_)) != FX_OK) return s;
    if ((s = fx_launch_derivative(c, g, 1, 2, 1.0, gg, 0.0, gy_)) != FX_OK) return s;
    {
        long long blocks = (n + 511) / 512;
        const long long cap = (long long)c->num_sms * 4;
        if (blocks > cap) blocks = cap;
        if (blocks < 1) blocks = 1;
        k_arakawa_products<<<(int)blocks, 512, 0, c->stream>>>(third, -third, f, gg, fx_, fy_, gx_, gy_, out, h1, h2, n);
        c->launches++;
        FX_CUDA(cudaGetLastError());
    }
    if ((s = fx_launch_derivative(c, g, 0, 2, 1.0, h1, 1.0, out)) != FX_OK) return s;                   // += Dx(...)
    return fx_launch_derivative(c, g, 1, 2, 1.0, h2, 1.0, out);                                         // += Dy(...)
}
extern "C" fx_status fx_arakawa(const fx_grid* g, const double* f, const double* gg, double* out) {
    FxCtx* c = fx_default_ctx();
    return c ? fx_arakawa_ex(c, g, f, gg, out) : FX_ECUDA;
}
