// fx_dgt.cuh -- the dG elliptic operator on a CTA-wide tile staged through shared memory by 2-D TMA.
//
// Paper: the derivative matrices have few distinct P x P blocks that must cost no memory traffic,
// P is a compile-time parameter, no divergent branches, fixed operation order with explicit FMAs
// (P:184-186); "higher polynomial order increases the registry pressure".
//
// The warp-strip kernel (fx_dg.cuh: one lane = one cell = P*P values of x, chi and the result in registers) runs into
// exactly that register wall on sm_100a: 8-12 warps per SM, issue/latency bound at 60-75 % of the HBM roofline.  Here no
// thread ever holds a cell.  A CTA owns a tile of TX = NBX*wb cells (wb <= 30) in x and marches through a segment of
// cell rows in y.  One elected lane moves every cell row (P image rows of x and chi, with a one-cell halo on each side:
// ONE box per vector) into a shared-memory ring with cp.async.bulk.tensor.2d (UTMALDG): out-of-range columns are
// zero-filled by the copy unit (the Dirichlet ghost); the periodic wrap-around is a separate one-cell box that only the
// first and last tile of a row load.  The operator is then evaluated by the same threads in two mappings per cell row:
//   * x-phase, one thread per (cell, image row): the P values of a line along x -- traces, gradient, flux, flux trace,
//     adjoint and jump of the x direction (DESIGN.md 3.4 steps 1-5) with constant-bank coefficients; neighbour-cell
//     traces travel by warp shuffle (lanes 1..wb produce, lanes 0 and wb+1 are the one-cell halo);
//   * y-phase, one thread per image column marching in y: the P values of the column in the cell row, traces carried in
//     registers from one step to the next; it receives the x-phase's (jx, sx) pair through a double-buffered
//     shared-memory hand-off, combines in the canonical order and stores the result with fully coalesced 8-byte stores.
// O(P) registers per thread instead of O(P*P); one __syncthreads per cell row; the loads cost no issue slots.
// Every intermediate still has the single defining expression of DESIGN.md 3.4, so the bits equal the oracle's and the
// warp-strip kernel's.

#ifndef FX_DGT_CUH
#define FX_DGT_CUH

#include <cuda.h>

#include "fx_dg.cuh"

#ifndef FX_NBX3
#define FX_NBX3 2
#endif
#ifndef FX_MINB3
#define FX_MINB3 3
#endif
#ifndef FX_NBX1
#define FX_NBX1 4
#endif
#ifndef FX_NBX4
#define FX_NBX4 1
#endif
#ifndef FX_NBX5
#define FX_NBX5 1
#endif
#ifndef FX_MINB4
#define FX_MINB4 3
#endif
#ifndef FX_MINB5
#define FX_MINB5 2
#endif
#ifndef FX_NS5
#define FX_NS5 4
#endif
#ifndef FX_KEEPP
#define FX_KEEPP 0        // keep the thread's table entries in registers for P <= FX_KEEPP (else they are re-read from the constant bank)
#endif
#define DGT_NS 4          // ring stages (cell rows resident or in flight per CTA) of the stand-alone apply
#ifndef FX_K1T_NS
#define FX_K1T_NS 4
#endif
#ifndef FX_K1T_R
#define FX_K1T_R 112
#endif
#ifndef FX_K1T_NBX
#define FX_K1T_NBX 2
#endif
#ifndef FX_K1T_ND
#define FX_K1T_ND 0
#endif
#ifndef FX_HPAD
#define FX_HPAD 1
#endif
#ifndef FX_XVEC
#define FX_XVEC 1
#endif
#define DGT_NS_K1 FX_K1T_NS   // ... of the fused CG kernel (three streams per stage)

// coefficient accessors of FX_CHAIN (fx_dg.cuh undefines its own at the end)
#define CL(m) g.L[m]
#define CR(m) g.R[m]
#define CB(m) g.B[m]
#define FF(m) f[m]

template <int P>
struct DgtCfg {
    static constexpr int NBX = P == 1 ? FX_NBX1 : P == 2 ? 2 : P == 3 ? FX_NBX3 : P == 4 ? FX_NBX4 : FX_NBX5;    // 30-cell x-blocks per CTA tile
    static constexpr int MINB = P == 5 ? FX_MINB5 : P == 4 ? FX_MINB4 : P == 3 ? FX_MINB3 : 3;   // CTAs per SM the register cap is sized for
    static constexpr int NS = P == 5 ? FX_NS5 : DGT_NS;                            // ring stages of the stand-alone apply
    static constexpr int NT = 32 * NBX * P;
    static constexpr int REGS = (65536 / (MINB * NT)) / 8 * 8 > 255 ? 255 : (65536 / (MINB * NT)) / 8 * 8;
};

template <int P, int NBX, int NSTR, int NS = DGT_NS, int ND = 0>
struct DgtGeom {
    static constexpr int TXM = FX_STRIP * NBX;                 // cells per tile at wb = 30
    static constexpr int SW = TXM * P;                         // doubles per image row of the tile proper (hand-off rows)
    static constexpr int HE = P & 1;                           // pad: boxes start at even columns (16-byte rule, see fx_dgt_shape)
    static constexpr int BW = (TXM + 2) * P + 2 * HE;          // main box: cells i0-1 .. i0+TXM, doubles per image row (even)
    static constexpr int HW = P + HE;                          // wrap box: one cell (even)
    static constexpr int MAIN_D = (P * BW * 8 + 127) / 128 * 16;   // doubles per region, 128-byte granules
    static constexpr int WRAP_D = (P * HW * 8 + 127) / 128 * 16;
    static constexpr int STR_D = MAIN_D + 2 * WRAP_D;          // one stream of one stage: main box, left wrap, right wrap
    static constexpr int STG_D = NSTR * STR_D;
    static constexpr int NTS = 32 * NBX * P;                    // stencil threads
    static constexpr int NT = NTS + 32 * (ND > 0 ? ND : 0);      // ... plus the exact-dot warps of the fused CG kernel (ND < 0: none, see dgt_tile)
    static constexpr unsigned MAIN_BYTES = (unsigned)(P * BW * 8), WRAP_BYTES = (unsigned)(P * HW * 8);
    // hand-off tile: cell pitch HP double2.  The x-phase lanes (one cell each) store P double2 at a stride of HP * 16 bytes:
    // 64 bytes (P = 4) would put the 8 lanes of a quarter-warp on 2 of the 8 16-byte bank groups (4-way conflict); 80 does not
    static constexpr int HP = (P == 4 && FX_HPAD) ? 5 : P;
    static constexpr int HSW = TXM * HP;                       // double2 per image row of the hand-off tile
    static constexpr size_t SMEM = (size_t)NS * STG_D * 8 + (size_t)2 * P * HSW * 16 * (ND != 0 ? 2 : 1);
};

struct DgtTile {                 // launch geometry of the tile kernels (host: fx_dgt_shape)
    int wb, ntx, rows_per_seg, nseg;
};

__device__ __forceinline__ void fx_tma_load_2d(unsigned dst, const CUtensorMap* map, int c0, int c1, unsigned bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"((unsigned long long)map), "r"(c0), "r"(c1), "r"(bar) : "memory");
}
__device__ __forceinline__ void fx_tma_prefetch_desc(const CUtensorMap* map) {
    asm volatile("prefetch.tensormap [%0];" ::"l"((unsigned long long)map) : "memory");
}

// ---- x lines of one (cell, image row): DESIGN.md 3.4 steps 1-5 along x ---------------------------------------------------
// u, c: the line's P values of the vector and of RN(WW*chi).  Results jx[k], sx[k].
// EDGE: this warp holds a ghost lane or a cell with a wall table (warp-uniform): only then are the selects compiled in.
template <int P, bool EDGE, bool NEU>
__device__ __forceinline__ void dgt_xline(const DgParams& g, const double (&u)[P], const double (&c)[P], bool xghost, bool firstx,
                                          bool lastx, bool mirlx, double (&jx)[P], double (&sx)[P]) {
    double tL, tR;
#define UU(m) u[m]
    FX_CHAIN(tL, CL, UU)
    FX_CHAIN(tR, CR, UU)
    if (EDGE && xghost) { tL = 0.0; tR = 0.0; }
    const double tLr = __shfl_down_sync(0xffffffffu, tL, 1), tRl = __shfl_up_sync(0xffffffffu, tR, 1);
    double f[P];
#pragma unroll
    for (int k = 0; k < P; ++k) {
        double a;
#define CT(m) dg_coef<EDGE, NEU>(g.T0[k][m], g.T0L[k][m], g.TD[k][m], firstx, lastx)
        FX_CHAIN(a, CT, UU)
#undef CT
        f[k] = __dmul_rn(c[k], __fma_rn(g.B[k], tLr, a));
    }
#undef UU
    double tB;
    FX_CHAIN(tB, CB, FF)
    if (EDGE && xghost) tB = 0.0;
    const double tBl = __shfl_up_sync(0xffffffffu, tB, 1);
    // the jump's ghost at a Neumann wall is the cell's own trace (difference +0); the gradient's ghost stays 0
    const double gxp = (EDGE && NEU) ? fx_selp(mirlx, tL, tRl) : tRl, gxn = (EDGE && NEU) ? fx_selp(lastx, tR, tLr) : tLr;
    const double dl = __dsub_rn(tL, gxp), dr = __dsub_rn(tR, gxn);
#pragma unroll
    for (int k = 0; k < P; ++k) {
        double a;
#define CT(m) dg_coef<EDGE, NEU>(g.T0[m][k], g.T0L[m][k], g.TD[m][k], firstx, lastx)
        FX_CHAIN(a, CT, FF)
#undef CT
        sx[k] = __fma_rn(g.L[k], tBl, a);
        jx[k] = __fma_rn(g.L[k], dl, __dmul_rn(g.R[k], dr));
    }
}

// ---- y lines of one image column in one cell row: flux, flux trace, adjoint (TK as in dg_ylines) -------------------------
template <int P, int TK>
__device__ __forceinline__ void dgt_yline(const DgParams& g, const double (&uc)[P], const double (&cc)[P], double tLyn, double tByp,
                                          double& tB, double (&sy)[P]) {
    double f[P];
#pragma unroll
    for (int l = 0; l < P; ++l) {
        double a;
#define UC(m) uc[m]
#define CT(m) (TK == 1 ? g.T0L[l][m] : TK == 2 ? g.TD[l][m] : g.T0[l][m])
        FX_CHAIN(a, CT, UC)
#undef CT
#undef UC
        f[l] = __dmul_rn(cc[l], __fma_rn(g.B[l], tLyn, a));
    }
    FX_CHAIN(tB, CB, FF)
#pragma unroll
    for (int l = 0; l < P; ++l) {
        double a;
#define CT(m) (TK == 1 ? g.T0L[m][l] : TK == 2 ? g.TD[m][l] : g.T0[m][l])
        FX_CHAIN(a, CT, FF)
#undef CT
        sy[l] = __fma_rn(g.L[l], tByp, a);
    }
}

template <bool B> struct DgtTag { static constexpr bool value = B; };
__device__ __forceinline__ void fx_keep(double& v) { asm volatile("" : "+d"(v)); }     // pin a loop-invariant in a register

// DIRF (the CG's fused direction update): the vector is p_new = fma(1, RN(V*r), RN(beta*p_old)) -- axpby(1, z,
// beta, p) with z = V o r in the canonical order of DESIGN.md 3.2 -- formed in shared memory from the staged rows of r and
// p_old by every thread that reads an element, stored to `pout` once per element, or p_old itself while upd is
// false (first iteration: p = z was set up by the caller).
struct DgtDir {
    const CUtensorMap *mr, *mrh;   // r: main and wrap boxes
    double* pout;
    double beta;
    bool upd;
};

// One CTA: tile `tx` of the cell columns, cell rows [j0, j1).  FUSE: feed the produced (x, y) pairs into the exact-dot
// accumulator `acc` (CG's p.Sp).  Shared memory: NS stages of {vector, chi [, r]} rows, then the hand-off double2[2][P][SW].
//
// Schedule.  Sequence number q = 0 .. n+1 is cell row j0 - 1 + q (q = 0: the row below the segment, whose top trace and
// flux trace enter the first row; q = n+1: the row above, of which only the bottom trace is needed; either is absent at a
// wall).  Iteration it = 0 .. n waits for q = it+1, runs the x-phase of that row (it < n) and the y-phase of row q = it
// (which needs the vector of row it+1 for the ghost trace and the x-phase results of the PREVIOUS iteration), then one
// __syncthreads; after it one lane refills the stage that iteration released -- the warps take turns, so that none of
// them is the straggler of every barrier.  Iterations 2 .. n-1 are "steady": no wall, no missing row, interior table --
// they run from a branch-free body, two per loop trip with the carried row alternating between two register sets.
// ND > 0 (with FUSE): the accumulation is done by ND warps of their own.  The column threads hand every (p, q) pair over
// through a second double-buffered shared-memory tile; the dot warps consume the pairs of iteration it-1 while the stencil
// warps work on iteration it.  (With the accumulator inside the column threads -- 19 registers of state, 23 fp64 and ~15
// other instructions per element inlined into the stencil code -- K1 spilled at 96 registers and ran 108-134 us.)
template <int P, int NBX, int NS, bool FUSE, bool DIRF, bool NEU, class ACC, int ND = 0>
__device__ __forceinline__ void dgt_tile(const DgParams& g, const DgtTile& t, const CUtensorMap* mu, const CUtensorMap* muh,
                                         const CUtensorMap* mc, const CUtensorMap* mch, const DgtDir& dir, double* __restrict__ y,
                                         unsigned long long* bars, int tx, int seg, int plane, ACC* acc, ExShared* sh) {
    typedef DgtGeom<P, NBX, DIRF ? 3 : 2, NS, ND> G;
    constexpr int NW = NBX * P;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int Nx = g.Nx, Ny = g.Ny, pitch = Nx * P;
    const int txc = t.wb * NBX;                                     // cells of this tile
    const int i0 = tx * txc;
    const int j0 = seg * t.rows_per_seg;
    const int j1 = (j0 + t.rows_per_seg < Ny) ? j0 + t.rows_per_seg : Ny;
    const int n = j1 - j0;
    const bool wallx = NEU ? g.bcx != 0 : g.bcx == 1, wally = NEU ? g.bcy != 0 : g.bcy == 1;
    const bool has_pro = !(j0 == 0 && wally), has_top = !(j1 == Ny && wally);
    // (the dynamic shared array is indexed directly: through a pointer parameter every access paid a generic-window base
    // computation, and asm loads with memory clobbers kept the compiler from interleaving the two phases)
    extern __shared__ __align__(128) double dgt_smem[];
    double2* const dgt_h = reinterpret_cast<double2*>(dgt_smem + (size_t)NS * G::STG_D);
    const unsigned sbase = fx_smem_addr(dgt_smem), full0 = fx_smem_addr(bars);
    constexpr int HBUF = P * G::HSW;                                 // double2 per hand-off buffer
    double2* const dgt_pq = dgt_h + 2 * HBUF;                        // ND > 0: the (p, q) pairs for the dot warps, double2[2][P][SW]
    const int cR = (i0 + txc < Nx) ? i0 + txc : Nx;                  // the cell after the tile's last one
    const bool wrapL = i0 == 0 && !wallx, wrapR = cR >= Nx && !wallx;    // periodic edge tiles: the halo cell is a box of its own

    // ---- x-phase identity: (x block, image row of the cell row), lane = cell -------------------------------------------
    const int xb = warp % NBX, xl = warp / NBX;
    const int ci = i0 - 1 + t.wb * xb + lane;                        // this lane's cell column (may be outside)
    const bool outside = ci < 0 || ci >= Nx;
    const bool xghost = outside && (wallx || ci < -1 || ci > Nx);    // contributes zero traces
    const bool produce = lane >= 1 && lane <= t.wb && ci < Nx;
    const bool firstx = (NEU ? g.lox == 1 : wallx) && ci == 0;       // T0L instead of T0 along x
    const bool lastx = NEU && g.hix == 2 && ci == Nx - 1;            // TD instead of T0; the jump's ghost mirrors
    const bool mirlx = NEU && g.lox == 2 && ci == 0;
    const bool edge = __any_sync(0xffffffffu, firstx || lastx || xghost);   // warp-uniform
    int xa, hw;                                                      // shared indices: my line in stage 0, my hand-off slot
    {
        int cl = ci - i0;
        if (cl < -1 || cl > G::TXM) cl = 0;                          // lanes beyond the halo are never looked at
        xa = xl * G::BW + G::HE + (cl + 1) * P;
        if (wrapL && ci == -1) xa = G::MAIN_D + xl * G::HW + G::HE;
        if (wrapR && ci == Nx) xa = G::MAIN_D + G::WRAP_D + xl * G::HW;
        if (cl < 0 || cl >= G::TXM) cl = 0;
        hw = xl * G::HSW + cl * G::HP;
    }

    FX_ASSERT(xa >= 0 && xa + P <= G::STR_D && hw >= 0 && hw + P <= P * G::HSW);
    FX_ASSERT(n >= 1 && i0 >= 0 && i0 < Nx && ((i0 * P) & 1) == 0 && txc <= G::TXM);
    // ---- y-phase identity: one image column ------------------------------------------------------------------------------
    const int ycol = tid < G::SW ? tid : G::SW - 1;
    const bool yact = tid < txc * P && (long long)i0 * P + tid < pitch;
    const int yk = ycol % P;
    const int hcol = (ycol / P) * G::HP + yk;                       // this column in a hand-off row
    const int ya = G::HE + P + ycol;
    const int zrow = plane * Ny * P;                                // first image row of this plane in the stacked vectors
    double wwy[P], wwx[P], jyk = g.JY[yk];                           // this thread's table entries
#pragma unroll
    for (int l = 0; l < P; ++l) { wwy[l] = g.WW[l][yk]; wwx[l] = g.WW[xl][l]; }
    if (P <= FX_KEEPP) {
#pragma unroll
        for (int l = 0; l < P; ++l) { fx_keep(wwy[l]); fx_keep(wwx[l]); }
        fx_keep(jyk);
    }
    double* yp = y + ((long long)zrow + (long long)j0 * P) * pitch + (long long)i0 * P + tid;     // row of the next output (yact threads only)
    const long long prow = (long long)pitch;

    // ---- TMA producer -----------------------------------------------------------------------------------------------------
    const int colM = (i0 - 1) * P - G::HE;                           // even (fx_dgt_shape); left of the image: zeros
    auto present = [&](int q) { return q == 0 ? has_pro : q == n + 1 ? has_top : true; };
    auto issue = [&](int q) {                                        // sequence q: cell row j0 - 1 + q into stage q % NS
        int r = j0 - 1 + q;
        if (r < 0) r += Ny;
        if (r >= Ny) r -= Ny;
        r = zrow + r * P;
        const unsigned nstr = (q <= n ? 2u : 1u) + (DIRF ? 1u : 0u);  // the row above the segment needs no chi
        const unsigned bar = full0 + 8u * (q % NS);
        FX_ASSERT(q >= 0 && q <= n + 1 && r >= 0 && r + P <= g.Nz * Ny * P);
        if (!present(q)) { fx_mbar_arrive(bar); return; }            // a row beyond a wall: the phase completes empty
        const unsigned dst = sbase + (unsigned)(q % NS) * (unsigned)(G::STG_D * 8);
        fx_mbar_expect_tx(bar, nstr * (G::MAIN_BYTES + (wrapL ? G::WRAP_BYTES : 0u) + (wrapR ? G::WRAP_BYTES : 0u)));
#pragma unroll
        for (int sidx = 0; sidx < (DIRF ? 3 : 2); ++sidx) {
            if (sidx == 1 && q > n) continue;
            const CUtensorMap* mm = sidx == 0 ? mu : sidx == 1 ? mc : dir.mr;
            const CUtensorMap* mh = sidx == 0 ? muh : sidx == 1 ? mch : dir.mrh;
            const unsigned d = dst + (unsigned)(sidx * G::STR_D * 8);
            fx_tma_load_2d(d, mm, colM, r, bar);
            if (wrapL) fx_tma_load_2d(d + G::MAIN_D * 8, mh, (Nx - 1) * P - G::HE, r, bar);
            if (wrapR) fx_tma_load_2d(d + (G::MAIN_D + G::WRAP_D) * 8, mh, 0, r, bar);
        }
    };
    if (tid == 0) {
#pragma unroll 1
        for (int q = 0; q < NS && q <= n + 1; ++q) issue(q);
    }
    int next = NS, pw = 0;                                            // next sequence number to load; the warp whose turn it is

    // ---- DIRF: p_new is formed on the fly by whoever reads an element (the x-phase thread for its line, the y-phase thread
    // for its column: 3 redundant fp64 operations per unknown instead of a separate pass through shared memory), and stored
    // to pout by the column thread.  Streams of a stage: 0 = p_old, 1 = chi, 2 = r.
    double* pp = DIRF ? dir.pout + ((long long)zrow + (long long)j0 * P) * pitch + (long long)i0 * P + tid : nullptr;
    const bool upd = DIRF && dir.upd;
    const double beta = DIRF ? dir.beta : 0.0;
    auto pnew = [&](double po, double rr, double v) { return upd ? __fma_rn(1.0, __dmul_rn(v, rr), __dmul_rn(beta, po)) : po; };

    // ND < 0: the pairs go through the same tile, but the stencil threads themselves consume the tile of the previous iteration
    // (one column each) after their y-phase: the accumulator code sits outside the stencil's live ranges
    int ncols = txc * P;
    if ((long long)i0 * P + ncols > pitch) ncols = pitch - i0 * P;
    auto consume_self = [&](int buf) {
        const double2* const pq = dgt_pq + buf * HBUF;
        const bool in = tid < ncols;
        double xs[P], ys[P];
        bool act[P];
#pragma unroll
        for (int l = 0; l < P; ++l) {
            const double2 v = in ? pq[l * G::SW + ycol] : make_double2(0.0, 0.0);
            xs[l] = v.x; ys[l] = v.y; act[l] = in;
        }
        acc->template add<P>(xs, ys, act, sh);
    };
    if (ND > 0 && FUSE && warp >= NW) {                              // ---- the exact-dot warps (see above) ----------------------
        const int dt = tid - NW * 32;
        int ncol = txc * P;
        if ((long long)i0 * P + ncol > pitch) ncol = pitch - i0 * P;
        if (ncol < 0) ncol = 0;
        auto consume = [&](int buf) {
            const double2* const pq = dgt_pq + buf * HBUF;
#pragma unroll 1
            for (int c0 = 0; c0 < ncol; c0 += ND * 32) {
                const int c = c0 + dt;
                const bool in = c < ncol;
                double xs[P], ys[P];
                bool act[P];
#pragma unroll
                for (int l = 0; l < P; ++l) {
                    const double2 v = in ? pq[l * G::SW + c] : make_double2(0.0, 0.0);
                    xs[l] = v.x; ys[l] = v.y; act[l] = in;
                }
                if (c0 + ND * 32 <= ncol) acc->template add_all<P>(xs, ys, sh);
                else acc->template add<P>(xs, ys, act, sh);
            }
        };
#pragma unroll 1
        for (int it = 0; it <= n; ++it) {                             // the pairs of iteration it-1 while the stencil warps run iteration it
            if (it >= 2) consume((it - 1) & 1);
            __syncthreads();
        }
        consume(n & 1);
        return;
    }

    double ua[P], ca[P], ub[P], cb[P];                                // the carried cell row: alternating register sets
    double tLy = 0.0, tRyp = 0.0, tByp = 0.0;
#pragma unroll
    for (int l = 0; l < P; ++l) { ua[l] = 0.0; ca[l] = 0.0; }
    if (has_pro) {                                                    // the row below the segment: its state enters step 0
        fx_mbar_wait(full0, 0u);
#pragma unroll
        for (int l = 0; l < P; ++l) {
            ua[l] = dgt_smem[ya + l * G::BW];
            if (DIRF) ua[l] = pnew(ua[l], dgt_smem[2 * G::STR_D + ya + l * G::BW], g.V[l][yk]);
            ca[l] = __dmul_rn(wwy[l], dgt_smem[G::STR_D + ya + l * G::BW]);
        }
    }

    // one iteration: uc/cc = the carried row (read), un/cn = the row loaded now (written).  ST: steady (see above).
    auto step = [&](auto st, const int it, const double (&uc)[P], const double (&cc)[P], double (&un)[P], double (&cn)[P]) {
        constexpr bool ST = decltype(st)::value;
        const int q = it + 1;
        const bool have = ST || present(q);
        const double* const sq = dgt_smem + (q % NS) * G::STG_D;
        if (have) fx_mbar_wait(full0 + 8u * (q % NS), (unsigned)((q / NS) & 1));

        // ---- x-phase of cell row j0 + it -----------------------------------------------------------------------------
        if (ST || it < n) {
            double u[P], c[P], jx[P], sx[P];
            if constexpr ((P & 1) == 0 && FX_XVEC != 0) {             // even P: a cell's line is 16-byte aligned (xa even): LDS.128 halves
#pragma unroll                                                        // the wavefronts of the lane-per-cell stride (P * 8 bytes)
                for (int m = 0; m < P; m += 2) {
                    const double2 uv = *reinterpret_cast<const double2*>(sq + xa + m);
                    const double2 cv = *reinterpret_cast<const double2*>(sq + G::STR_D + xa + m);
                    u[m] = uv.x; u[m + 1] = uv.y;
                    if (DIRF) {
                        const double2 rv = *reinterpret_cast<const double2*>(sq + 2 * G::STR_D + xa + m);
                        u[m] = pnew(u[m], rv.x, g.V[xl][m]);
                        u[m + 1] = pnew(u[m + 1], rv.y, g.V[xl][m + 1]);
                    }
                    c[m] = __dmul_rn(wwx[m], cv.x); c[m + 1] = __dmul_rn(wwx[m + 1], cv.y);
                }
            } else {
#pragma unroll
                for (int m = 0; m < P; ++m) {
                    u[m] = sq[xa + m];
                    if (DIRF) u[m] = pnew(u[m], sq[2 * G::STR_D + xa + m], g.V[xl][m]);
                    c[m] = __dmul_rn(wwx[m], sq[G::STR_D + xa + m]);
                }
            }
            if (edge) dgt_xline<P, true, NEU>(g, u, c, xghost, firstx, lastx, mirlx, jx, sx);
            else dgt_xline<P, false, NEU>(g, u, c, xghost, firstx, lastx, mirlx, jx, sx);
            if (produce) {
                double2* const h = dgt_h + (it & 1) * HBUF + hw;
#pragma unroll
                for (int k = 0; k < P; ++k) h[k] = make_double2(jx[k], sx[k]);
            }
        }

        // ---- y-phase of cell row r = j0 - 1 + it ----------------------------------------------------------------------
        if (have) {
#pragma unroll
            for (int l = 0; l < P; ++l) un[l] = sq[ya + l * G::BW];
            if (DIRF) {
#pragma unroll
                for (int l = 0; l < P; ++l) un[l] = pnew(un[l], sq[2 * G::STR_D + ya + l * G::BW], g.V[l][yk]);
                if (ST || it < n) {                                   // rows j0 .. j1-1: this thread stores its column of p_new
                    if (yact) {
#pragma unroll
                        for (int l = 0; l < P; ++l) pp[l * prow] = un[l];
                    }
                    pp += P * prow;
                }
            }
            if (ST || it < n) {
#pragma unroll
                for (int l = 0; l < P; ++l) cn[l] = __dmul_rn(wwy[l], sq[G::STR_D + ya + l * G::BW]);
            }
        }
        double tLyn;
#define UN(m) un[m]
        FX_CHAIN(tLyn, CL, UN)
#undef UN
        if (!have) tLyn = 0.0;                                        // beyond a wall: zero ghost trace
        if (!ST && it == 0 && !has_pro) {                             // segment starts at a wall: no row below
            tLy = tLyn;
            tRyp = (NEU && g.loy == 2) ? tLy : 0.0;                   // Neumann: mirrored, jump +0
            tByp = 0.0;
        } else {
            int r = j0 - 1 + it;
            if (!ST && r < 0) r += Ny;
            double tRy, tB, sy[P];
#define UC(m) uc[m]
            FX_CHAIN(tRy, CR, UC)
#undef UC
            if (!ST && NEU && g.hiy == 2 && r == Ny - 1) dgt_yline<P, 2>(g, uc, cc, tLyn, tByp, tB, sy);
            else if (!ST && (NEU ? g.loy == 1 : wally) && r == 0) dgt_yline<P, 1>(g, uc, cc, tLyn, tByp, tB, sy);
            else dgt_yline<P, 0>(g, uc, cc, tLyn, tByp, tB, sy);
            if (ST || it >= 1) {
                const double gyn = (!ST && NEU && !have && g.hiy == 2) ? tRy : tLyn;
                const double dl = __dsub_rn(tLy, tRyp), dr = __dsub_rn(tRy, gyn);
                const double2* const h = dgt_h + ((it - 1) & 1) * HBUF + hcol;
                double o[P];
#pragma unroll
                for (int l = 0; l < P; ++l) {
                    const double2 hx = h[l * G::HSW];
                    const double jy = __fma_rn(g.L[l], dl, __dmul_rn(g.R[l], dr));
                    double v = __fma_rn(g.JX[l], hx.x, __dmul_rn(jyk, jy));
                    v = __fma_rn(g.cyy, sy[l], v);
                    v = __fma_rn(g.cxx, hx.y, v);
                    if (g.normed) v = __dmul_rn(g.V[l][yk], v);
                    else if (g.zmul) v = __dmul_rn(g.hz, v);
                    o[l] = v;
                }
                if (yact) {
#pragma unroll
                    for (int l = 0; l < P; ++l) yp[l * prow] = o[l];
                }
                yp += P * prow;
                if (FUSE && ND != 0) {                                // hand the pairs to the dot warps (or to the later self)
                    if (tid < G::SW) {
                        double2* const pq = dgt_pq + (it & 1) * HBUF + ycol;
#pragma unroll
                        for (int l = 0; l < P; ++l) pq[l * G::SW] = make_double2(uc[l], o[l]);
                    }
                } else if (FUSE) {
                    double xs[P], ys[P];
                    bool act[P];
#pragma unroll
                    for (int l = 0; l < P; ++l) { xs[l] = yact ? uc[l] : 0.0; ys[l] = yact ? o[l] : 0.0; act[l] = yact; }
                    acc->template add<P>(xs, ys, act, sh);
                }
            }
            tRyp = tRy; tByp = tB; tLy = tLyn;
        }
        if (FUSE && ND < 0 && (ST || it >= 2)) consume_self((it - 1) & 1);
        __syncthreads();
        // iteration `it` is over: the stages of q <= it+1 are free
        const int lim = (it + 1 + NS < n + 1) ? it + 1 + NS : n + 1;
        if (warp == pw && lane == 0)
            for (int qq = next; qq <= lim; ++qq) issue(qq);
        if (lim >= next) next = lim + 1;
        pw = (pw + 1 == NW) ? 0 : pw + 1;
    };
    auto generic = [&](int it) {                                      // in place: the carried row stays in set a
#pragma unroll
        for (int l = 0; l < P; ++l) { ub[l] = ua[l]; cb[l] = ca[l]; }
        step(DgtTag<false>(), it, ub, cb, ua, ca);
    };

    int it = 0;
    int pre = 2 + ((n > 2 && ((n - 2) & 1)) ? 1 : 0);                 // then an even number of steady iterations is left
    if (pre > n + 1) pre = n + 1;
#pragma unroll 1
    for (; it < pre; ++it) generic(it);
#pragma unroll 1
    for (; it + 1 <= n - 1; it += 2) {
        step(DgtTag<true>(), it, ua, ca, ub, cb);
        step(DgtTag<true>(), it + 1, ub, cb, ua, ca);
    }
#pragma unroll 1
    for (; it <= n; ++it) generic(it);
    if (FUSE && ND < 0) consume_self(n & 1);                          // (written in iteration n, before its barrier)
}

#undef CL
#undef CR
#undef CB
#undef FF

#endif
