// fx_dg.cuh -- the dG elliptic operator y = S x (or A x = V o S x) as one fused block-stencil kernel.
//
// Paper: the dG derivatives are block-sparse matrices with few distinct P x P blocks, kept out of the memory
// traffic so that the product is bandwidth bound like axpby; P is a compile-time
// parameter for tight inner loops; no divergent branches; fixed operation order with explicit
// FMAs for bitwise reproducibility.  The paper applies dx, dy and jump matrices one call at a time
// (6 mat-vecs per elliptic apply) and names that modularity a factor 2-5 loss.
//
// Here: ONE kernel reads x and chi once and writes y once (24 B per unknown).  A warp owns a
// strip of 30 cells in x (lanes 1..30; lanes 0 and 31 are the one-cell halo and recompute only traces and flux
// traces) and marches through a segment of cell rows in y.  A lane holds its cell's P*P values in registers.
// Everything that couples neighbouring cells is a *trace* (P numbers per cell side): in x they travel by warp
// shuffle, in y they are carried in registers from one marching step to the next.  No shared memory, no
// __syncthreads, no tensor cores (this is a bandwidth-bound stencil, not a dense contraction).
// The operation sequence per node is exactly DESIGN.md 3.4; every intermediate has a single defining
// expression, so halo recomputation and any launch shape give the same bits.

#ifndef FX_DG_CUH
#define FX_DG_CUH

#include "fx_exdot.cuh"
#include "fx_stream.cuh"
#include "fx_tables.h"

struct DgParams {
    int Nx, Ny, bcx, bcy;          // fx_bc of each direction
    int lox, hix, loy, hiy;        // the four walls: 0 = none (periodic), 1 = Dirichlet, 2 = Neumann
    int rows_per_seg, nseg, nstrip;
    int normed;
    int smr;                       // rows staged through the per-lane shared-memory ring (P <= 3)
    int Nz, zmul;                  // 3-D product grid (Q24): planes stacked in the vectors; zmul: (S x) is multiplied by hz
    double hz;
    double cxx, cyy;               // hy/hx, hx/hy
    double T0[FX_PMAX][FX_PMAX], T0L[FX_PMAX][FX_PMAX], WW[FX_PMAX][FX_PMAX], V[FX_PMAX][FX_PMAX];
    double TD[FX_PMAX][FX_PMAX];   // D: the cell table of the last cell before a Neumann wall
    double B[FX_PMAX], L[FX_PMAX], R[FX_PMAX], JX[FX_PMAX], JY[FX_PMAX];
};

#define FX_STRIP 30
#ifndef FX_PFD
#define FX_PFD 1          // prefetch distance in marching steps (2 and 3 measured slower: L1 capacity / set conflicts)
#endif

template <int P>
struct DgCell { double v[P][P]; };     // [l][k]: row l (y node), column k (x node)

// load one cell's P x P values (always from valid memory: ghost lanes read their wrapped cell and have their traces
// forced to +0.0 afterwards, which is all their neighbours ever see)
// COH: the array is rewritten by this very kernel (the persistent CG loop, between grid syncs): the non-coherent path
// (ld.global.nc) is only defined for data that stays read-only for the whole kernel, so such arrays are read with
// ld.global.cg (L2, where the grid sync made the new values visible) and are not prefetched into L1.
template <int P, bool COH = false>
__device__ __forceinline__ void dg_load(DgCell<P>& c, const double* a, long long pitch, int col0, int j,
                                        bool) {
    const double* q = a + (long long)j * P * pitch + col0;
#pragma unroll
    for (int l = 0; l < P; ++l)
#pragma unroll
        for (int k = 0; k < P; ++k) c.v[l][k] = COH ? __ldcg(q + l * pitch + k) : __ldg(q + l * pitch + k);
}

// L1 prefetch of one cell (the first element of each of its P rows; a lane's P doubles span at most two 32-byte
// sectors and the neighbouring lane touches the second one)
template <int P>
__device__ __forceinline__ void dg_prefetch(const double* __restrict__ a, long long pitch, int col0, int j) {
    const double* q = a + (long long)j * P * pitch + col0;
#pragma unroll
    for (int l = 0; l < P; ++l) asm volatile("prefetch.global.L1 [%0];" ::"l"(q + l * pitch));
}

// Source of the vector the operator is applied to.  DIRF (the CG's fused direction update): the vector is
// p_new = fma(1, RN(V*r), RN(beta*p_old)) formed on the fly from r and p_old -- axpby(1, z, beta, p) with z = V o r in
// the canonical order of DESIGN.md 3.2 -- or p_old itself while upd is false (first iteration: p = z was set up).
struct DgSrc {
    const double* x;       // the vector (DIRF: p_old)
    const double* r;       // DIRF only
    double* pout;          // DIRF only: where p_new is stored (a different buffer than x: neighbours still read p_old)
    double beta;
    bool upd;
};

template <int P, bool DIRF, bool COH = false>
__device__ __forceinline__ void dg_load_u(DgCell<P>& c, const DgParams& g, const DgSrc& s, long long pitch, int col0, int j) {
    dg_load<P, COH>(c, s.x, pitch, col0, j, false);
    if (DIRF) {
        if (s.upd) {
            DgCell<P> rr;
            dg_load<P, COH>(rr, s.r, pitch, col0, j, false);
#pragma unroll
            for (int l = 0; l < P; ++l)
#pragma unroll
                for (int k = 0; k < P; ++k)
                    c.v[l][k] = __fma_rn(1.0, __dmul_rn(g.V[l][k], rr.v[l][k]), __dmul_rn(s.beta, c.v[l][k]));
        }
    }
}

// ---- per-lane shared-memory row ring (SMR path, P <= 3) -------------------------------------------------------------------
// The generic path above relies on L1 prefetches; rows of one cell lie one image row (a multiple of 8 KB at the
// benchmark sizes) apart, so they compete for the same L1 sets and ~1/3 of the register loads still miss.  With SMR every
// lane copies ITS OWN cell of the rows ahead into its own shared-memory slots with cp.async (as the streaming kernels do,
// fx_stream.cuh) and reads them back after cp.async.wait_group: residency is guaranteed, no barrier, no extra registers.
// Slot = P*P doubles per lane, lane-interleaved (conflict-free); slots 0..2: input vector rows (sequence number mod 3),
// 3..4: chi (mod 2), 5..7: r for the fused direction update.
template <int P>
__device__ __forceinline__ void smr_issue(double* ring, int slot, const double* __restrict__ a, long long pitch, int col0, int jr) {
    const double* q = a + (long long)jr * P * pitch + col0;
    FX_ASSERT(slot >= 0 && slot < 8 && jr >= 0 && col0 >= 0 && col0 + P <= pitch);      // own slot of the ring, a row of the image
    const unsigned dst = fx_smem_addr(ring + (size_t)slot * P * P * 32 + (threadIdx.x & 31));
#pragma unroll
    for (int l = 0; l < P; ++l)
#pragma unroll
        for (int k = 0; k < P; ++k) fx_cp_async8(dst + (unsigned)((l * P + k) * 32 * 8), q + l * pitch + k, true);
}
template <int P>
__device__ __forceinline__ void smr_read(DgCell<P>& c, const double* ring, int slot) {
    const double* q = ring + (size_t)slot * P * P * 32 + (threadIdx.x & 31);
#pragma unroll
    for (int l = 0; l < P; ++l)
#pragma unroll
        for (int k = 0; k < P; ++k) c.v[l][k] = q[(l * P + k) * 32];
}
template <int P, bool DIRF>
__device__ __forceinline__ void smr_read_u(DgCell<P>& c, const DgParams& g, const DgSrc& s, const double* ring, int sq) {
    smr_read<P>(c, ring, sq % 3);
    if (DIRF && s.upd) {
        DgCell<P> rr;
        smr_read<P>(rr, ring, 5 + sq % 3);
#pragma unroll
        for (int l = 0; l < P; ++l)
#pragma unroll
            for (int k = 0; k < P; ++k)
                c.v[l][k] = __fma_rn(1.0, __dmul_rn(g.V[l][k], rr.v[l][k]), __dmul_rn(s.beta, c.v[l][k]));
    }
}

// chain over m:  acc = c[0]*v[0]; acc = fma(c[m], v[m], acc)
#define FX_CHAIN(acc, COEF, VAL)                         \
    {                                                    \
        acc = __dmul_rn(COEF(0), VAL(0));                \
        _Pragma("unroll") for (int m_ = 1; m_ < P; ++m_) \
            acc = __fma_rn(COEF(m_), VAL(m_), acc);      \
    }
#define CL(m) g.L[m]
#define CR(m) g.R[m]
#define CB(m) g.B[m]
#define FF(m) f[m]

// y lines of one cell: flux, flux trace, adjoint; acc_ += cyy * sy.  TK: the cell table -- 0 = T0, 1 = T0L (first cell
// of a line that starts at a Dirichlet wall), 2 = TD (last cell of a line that ends at a Neumann wall).
// tByp: in = flux trace of the cell below, out = this cell's.  The P*P chains of each stage are independent: they are
// written stage by stage so that the scheduler sees P*P-way instruction-level parallelism.
template <int P, int TK>
__device__ __forceinline__ void dg_ylines(const DgParams& g, const DgCell<P>& uc, const DgCell<P>& cc, const double (&tLyn)[P],
                                          double (&tByp)[P], double (&acc_)[P][P]) {
    double f[P][P];                                                   // f[l][k]
#pragma unroll
    for (int l = 0; l < P; ++l)
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double a;
#define UC(m) uc.v[m][k]
#define CT(m) (TK == 1 ? g.T0L[l][m] : TK == 2 ? g.TD[l][m] : g.T0[l][m])
            FX_CHAIN(a, CT, UC)
#undef CT
#undef UC
            f[l][k] = __dmul_rn(cc.v[l][k], __fma_rn(g.B[l], tLyn[k], a));
        }
    double tB[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {
#define FK(m) f[m][k]
        FX_CHAIN(tB[k], CB, FK)
    }
#pragma unroll
    for (int l = 0; l < P; ++l)
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double a;
#define CT(m) (TK == 1 ? g.T0L[m][l] : TK == 2 ? g.TD[m][l] : g.T0[m][l])
            FX_CHAIN(a, CT, FK)
#undef CT
            acc_[l][k] = __fma_rn(g.cyy, __fma_rn(g.L[l], tByp[k], a), acc_[l][k]);
        }
#undef FK
#pragma unroll
    for (int k = 0; k < P; ++k) tByp[k] = tB[k];
}

// Cell-table coefficient of this lane's cell along x.  Periodic / Dirichlet: one two-way select.  With Neumann walls the
// three-way choice is spelled as two selp (as plain conditionals the compiler turns it into divergent branches around
// every FMA, and the two wall strips then take twice as long as the rest of the single wave).
__device__ __forceinline__ double fx_selp(bool c, double a, double b) {
    double r;
    asm("{\n\t.reg .pred p;\n\tsetp.ne.s32 p, %3, 0;\n\tselp.f64 %0, %1, %2, p;\n\t}" : "=d"(r) : "d"(a), "d"(b), "r"((int)c));
    return r;
}
template <bool SEL, bool NEU>
__device__ __forceinline__ double dg_coef(double t0, double t0l, double td, bool firstx, bool lastx) {
    if (!SEL) return t0;
    if (!NEU) return firstx ? t0l : t0;
    return fx_selp(lastx, td, fx_selp(firstx, t0l, t0));
}

// x lines of one cell.  SEL: this warp contains a cell with a wall table (lane flags firstx: T0L; lastx, NEU only: TD).
// out[l][k] = cxx * sx + acc_ (times V if normed)
template <int P, bool SEL, bool NEU>
__device__ __forceinline__ void dg_xlines(const DgParams& g, const DgCell<P>& uc, const DgCell<P>& cc, const double (&tLxr)[P],
                                          bool firstx, bool lastx, bool xghost, double (&acc_)[P][P]) {
    double f[P][P];                                                   // f[l][k]
#pragma unroll
    for (int l = 0; l < P; ++l)
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double a;
#define UC(m) uc.v[l][m]
#define CT(m) dg_coef<SEL, NEU>(g.T0[k][m], g.T0L[k][m], g.TD[k][m], firstx, lastx)
            FX_CHAIN(a, CT, UC)
#undef CT
#undef UC
            f[l][k] = __dmul_rn(cc.v[l][k], __fma_rn(g.B[k], tLxr[l], a));
        }
    double tBl[P];
#pragma unroll
    for (int l = 0; l < P; ++l) {
        double tB;
#define FL(m) f[l][m]
        FX_CHAIN(tB, CB, FL)
        if (xghost) tB = 0.0;
        tBl[l] = __shfl_up_sync(0xffffffffu, tB, 1);
    }
#pragma unroll
    for (int l = 0; l < P; ++l)
#pragma unroll
        for (int k = 0; k < P; ++k) {
            double a;
#define CT(m) dg_coef<SEL, NEU>(g.T0[m][k], g.T0L[m][k], g.TD[m][k], firstx, lastx)
            FX_CHAIN(a, CT, FL)
#undef CT
            double o = __fma_rn(g.cxx, __fma_rn(g.L[k], tBl[l], a), acc_[l][k]);
            if (g.normed) o = __dmul_rn(g.V[l][k], o);
            else if (g.zmul) o = __dmul_rn(g.hz, o);
            acc_[l][k] = o;
        }
#undef FL
}

// One warp: strip `strip` of 30 cells, cell rows [j0, j1).  FUSE: feed (x, y) pairs of the produced cells into the
// exact-dot accumulator `acc` (the CG's p.Sp).
// NEU: the grid has a Neumann wall (a separate instantiation, so that the periodic / Dirichlet code is untouched by it).
template <int P, bool FUSE, bool DIRF, bool SMR, bool NEU, class ACC, bool COH = false>
__device__ __forceinline__ void dg_warp_strip(const DgParams& g, const double* __restrict__ chi, const DgSrc& src,
                                              double* __restrict__ y, int strip, int j0, int j1, ACC* acc, ExShared* sh,
                                              double* ring) {
    const double* x = src.x;
    const int lane = threadIdx.x & 31;
    const int Nx = g.Nx, Ny = g.Ny;
    const long long pitch = (long long)Nx * P;
    const int ci = strip * FX_STRIP - 1 + lane;                    // this lane's cell column (may be outside)
    const bool outside = ci < 0 || ci >= Nx;
    const bool dirx = NEU ? g.bcx != 0 : g.bcx == 1, diry = NEU ? g.bcy != 0 : g.bcy == 1;   // walls (ghost traces are zero)
    // periodic: wrap once; lanes further out are never used but must read valid memory
    int cw = ci;
    if (outside) { cw = ci % Nx; if (cw < 0) cw += Nx; }
    const bool xghost = outside && (dirx || ci < -1 || ci > Nx);   // contributes zero traces
    const bool produce = lane >= 1 && lane <= FX_STRIP && ci < Nx; // ci >= 0 holds for lanes >= 1
    const bool firstx = (NEU ? g.lox == 1 : dirx) && ci == 0;      // T0L instead of T0 along x
    const bool lastx = NEU && g.hix == 2 && ci == Nx - 1;          // TD instead of T0 along x; the jump's ghost mirrors
    const bool mirlx = NEU && g.lox == 2 && ci == 0;               // lower Neumann wall: the jump's ghost mirrors
    const bool selx = dirx && (strip == 0 || (NEU && strip == g.nstrip - 1));   // warp-uniform: some lane has a wall table
    const int col0 = cw * P;
    FX_ASSERT(cw >= 0 && cw < Nx && j0 >= 0 && j0 < j1 && j1 <= Ny);

    DgCell<P> uc, un, cc;
    double tLy[P], tRyp[P], tByp[P];                               // own bottom trace; previous cell's top / flux trace

    // ---- prologue: state of cell row j0-1 ------------------------------------------------------------------
    dg_load_u<P, DIRF, COH>(uc, g, src, pitch, col0, j0);
    dg_load<P>(cc, chi, pitch, col0, j0, xghost);
    // L1 prefetch, FX_PFD steps ahead: row jr of the input vector (needed as the upper neighbour at step jr-1) and of chi
    auto pf_x = [&](int jr) {
        if (COH || xghost || jr > j1) return;
        if (jr >= Ny) { if (diry) return; jr -= Ny; }
        dg_prefetch<P>(x, pitch, col0, jr); if (DIRF) dg_prefetch<P>(src.r, pitch, col0, jr);
    };
    auto pf_c = [&](int jr) { if (!xghost && jr < j1) dg_prefetch<P>(chi, pitch, col0, jr); };
    auto rowx = [&](int jr) { return jr >= Ny ? jr - Ny : jr; };       // beyond the top: wrap (a Dirichlet ghost row is never used)
    if (SMR) {
        smr_issue<P>(ring, 1, x, pitch, col0, rowx(j0 + 1));
        if (DIRF) smr_issue<P>(ring, 5 + 1, src.r, pitch, col0, rowx(j0 + 1));
        fx_cp_commit();
    } else {
#pragma unroll
        for (int d = 1; d <= FX_PFD; ++d) { pf_x(j0 + d); pf_c(j0 + d); }
    }
#pragma unroll
    for (int k = 0; k < P; ++k) {
#define UC(m) uc.v[m][k]
        FX_CHAIN(tLy[k], CL, UC)
#undef UC
    }
    if (j0 == 0 && diry) {
#pragma unroll
        for (int k = 0; k < P; ++k) { tRyp[k] = (NEU && g.loy == 2) ? tLy[k] : 0.0; tByp[k] = 0.0; }   // Neumann: mirrored, jump +0
    } else {
        const int jp = (j0 == 0) ? Ny - 1 : j0 - 1;
        DgCell<P> up, cp;
        dg_load_u<P, DIRF, COH>(up, g, src, pitch, col0, jp);
        dg_load<P>(cp, chi, pitch, col0, jp, xghost);
        double dummy[P][P];
#pragma unroll
        for (int k = 0; k < P; ++k) {
#define UP(m) up.v[m][k]
            FX_CHAIN(tRyp[k], CR, UP)
#undef UP
            tByp[k] = 0.0;
#pragma unroll
            for (int l = 0; l < P; ++l) { cp.v[l][k] = __dmul_rn(g.WW[l][k], cp.v[l][k]); dummy[l][k] = 0.0; }
        }
        if ((NEU ? g.loy == 1 : diry) && jp == 0) dg_ylines<P, 1>(g, up, cp, tLy, tByp, dummy);
        else dg_ylines<P, 0>(g, up, cp, tLy, tByp, dummy);
    }

    // ---- march ---------------------------------------------------------------------------------------------
    // Every cell row is fetched from HBM once, by an L1 prefetch one step ahead; the register loads below are L1
    // hits.  u of a row is read twice (as the row above, for its bottom trace, then as the current row): holding it
    // in registers across the step instead costs 2*P*P registers and a quarter of the occupancy.
    for (int j = j0; j < j1; ++j) {
        int jn = j + 1;
        bool yghost = false;
        if (jn == Ny) { jn = 0; yghost = diry; }
        if (SMR) {
            const int sq = j - j0;
            if (j + 1 < j1) {                                        // the rows of the next step
                smr_issue<P>(ring, (sq + 2) % 3, x, pitch, col0, rowx(j + 2));
                if (DIRF) smr_issue<P>(ring, 5 + (sq + 2) % 3, src.r, pitch, col0, rowx(j + 2));
                smr_issue<P>(ring, 3 + ((sq + 1) & 1), chi, pitch, col0, j + 1);
            }
            fx_cp_commit();
            fx_cp_wait<1>();                                         // everything but the group just committed has landed
            if (j > j0) { if (!DIRF) smr_read_u<P, DIRF>(uc, g, src, ring, sq); smr_read<P>(cc, ring, 3 + (sq & 1)); }
            smr_read_u<P, DIRF>(un, g, src, ring, sq + 1);
        } else {
            if (j > j0) { if (!DIRF) dg_load_u<P, DIRF, COH>(uc, g, src, pitch, col0, j); dg_load<P>(cc, chi, pitch, col0, j, xghost); }
            dg_load_u<P, DIRF, COH>(un, g, src, pitch, col0, jn);
            pf_x(j + 1 + FX_PFD); pf_c(j + FX_PFD);                // rows of the steps ahead
        }

        double tRy[P], tLyn[P], tLx[P], tRx[P];
#pragma unroll
        for (int k = 0; k < P; ++k) {
#define UC(m) uc.v[m][k]
#define UN(m) un.v[m][k]
            FX_CHAIN(tRy[k], CR, UC)
            FX_CHAIN(tLyn[k], CL, UN)
            if (yghost) tLyn[k] = 0.0;
#undef UC
#undef UN
        }
#pragma unroll
        for (int l = 0; l < P; ++l) {
#define UC(m) uc.v[l][m]
            FX_CHAIN(tLx[l], CL, UC)
            FX_CHAIN(tRx[l], CR, UC)
#undef UC
            if (xghost) { tLx[l] = 0.0; tRx[l] = 0.0; }
        }
        // c = RN(WW * chi), jumps first (DESIGN.md 3.4 combine order: JY*jy, then + JX*jx, + cyy*sy, + cxx*sx)
        double acc_[P][P];
        double tLxr[P], tRxl[P];
#pragma unroll
        for (int l = 0; l < P; ++l) {
            tLxr[l] = __shfl_down_sync(0xffffffffu, tLx[l], 1);
            tRxl[l] = __shfl_up_sync(0xffffffffu, tRx[l], 1);
        }
#pragma unroll
        for (int l = 0; l < P; ++l)
#pragma unroll
            for (int k = 0; k < P; ++k) {
                cc.v[l][k] = __dmul_rn(g.WW[l][k], cc.v[l][k]);
                // the jump's ghost at a Neumann wall is the cell's own trace (difference +0); the gradient's ghost stays 0
                const double gyn = (NEU && yghost && g.hiy == 2) ? tRy[k] : tLyn[k];
                const double gxp = NEU ? fx_selp(mirlx, tLx[l], tRxl[l]) : tRxl[l], gxn = NEU ? fx_selp(lastx, tRx[l], tLxr[l]) : tLxr[l];
                const double jy = __fma_rn(g.L[l], __dsub_rn(tLy[k], tRyp[k]), __dmul_rn(g.R[l], __dsub_rn(tRy[k], gyn)));
                const double jx = __fma_rn(g.L[k], __dsub_rn(tLx[l], gxp), __dmul_rn(g.R[k], __dsub_rn(tRx[l], gxn)));
                acc_[l][k] = __fma_rn(g.JX[l], jx, __dmul_rn(g.JY[k], jy));
            }
        if (NEU && g.hiy == 2 && j == Ny - 1) dg_ylines<P, 2>(g, uc, cc, tLyn, tByp, acc_);
        else if ((NEU ? g.loy == 1 : diry) && j == 0) dg_ylines<P, 1>(g, uc, cc, tLyn, tByp, acc_);
        else dg_ylines<P, 0>(g, uc, cc, tLyn, tByp, acc_);
#pragma unroll
        for (int k = 0; k < P; ++k) { tRyp[k] = tRy[k]; tLy[k] = tLyn[k]; }
        if (selx) dg_xlines<P, true, NEU>(g, uc, cc, tLxr, firstx, lastx, xghost, acc_);
        else dg_xlines<P, false, NEU>(g, uc, cc, tLxr, firstx, lastx, xghost, acc_);

        if (DIRF && produce) {
            double* prow = src.pout + (long long)j * P * pitch + col0;
#pragma unroll
            for (int l = 0; l < P; ++l)
#pragma unroll
                for (int k = 0; k < P; ++k) prow[l * pitch + k] = uc.v[l][k];
        }
        if (produce) {
            double* yrow = y + (long long)j * P * pitch + col0;
#pragma unroll
            for (int l = 0; l < P; ++l)
#pragma unroll
                for (int k = 0; k < P; ++k) yrow[l * pitch + k] = acc_[l][k];
        }
        if (FUSE) {
            double xs[P * P], ys[P * P];
            bool act[P * P];
#pragma unroll
            for (int l = 0; l < P; ++l)
#pragma unroll
                for (int k = 0; k < P; ++k) {
                    xs[l * P + k] = produce ? uc.v[l][k] : 0.0; ys[l * P + k] = produce ? acc_[l][k] : 0.0; act[l * P + k] = produce;
                }
            acc->template add<P * P>(xs, ys, act, sh);
        }
        if (DIRF) uc = un;                                           // formed once per row: carried instead of re-formed
    }
    if (SMR) fx_cp_wait<0>();
}
#undef CL
#undef CR
#undef CB
#undef FF

#endif
