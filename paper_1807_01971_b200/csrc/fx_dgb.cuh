// fx_dgb.cuh -- the Arakawa bracket in two kernels on the CTA-tile stencil of fx_dgt.cuh.
//
// Paper: the bracket is benchmarked as N = 9 calls with M = 34 vector passes; "with a fused implementation" N = 1, M = 4
// would do (Fig. 6a).  The nine calls: four centred derivatives f_x, f_y, g_x, g_y; three
// fused products out = 1/3 (f_x g_y - f_y g_x), h1 = 1/3 (f g_y - g f_y), h2 = 1/3 (g f_x - f g_x); out += D_x h1; out += D_y h2.
// Here (same operations in the same order, the same bits):
//   stage A  reads f, g (with halos), forms the four derivatives on the fly -- the x derivatives by the (cell, image row)
//            threads, the y derivatives by the image-column threads, (f_x, g_x) crossing through the shared-memory hand-off --
//            and writes out, h1, h2:                              2 + 3 = 5 vector passes;
//   stage B  reads h1, h2, out, forms D_x h1 (row threads) and D_y h2 (column threads), writes out = RN(D_y h2 + RN(D_x h1 + out)):
//                                                                  3 + 1 = 4 vector passes.
// A single kernel cannot do it: D_x h1 at a node needs h1 of the whole x-line of its cell and of both neighbour cells, and h1
// needs f_y, g_y there, i.e. a two-cell halo recomputed in both directions; the honest floor with halo recompute is M = 5-6,
// two kernels give 9 against the 23 of the seven launches they replace.
// Centred derivative of a line, cell n, node k:  a = chain_m(TT[k][m], u_{n,m});  a = fma(cP[k], tR_{n-1}, a);
// a = fma(cN[k], tL_{n+1}, a);  d = RN(s * a), s = 2/h;  with alpha = 1, beta = 0 the call's result is d itself.

#ifndef FX_DGB_CUH
#define FX_DGB_CUH

#include "fx_dgt.cuh"

struct DbParams {
    int Nx, Ny, bcx, bcy;                          // PER or DIR
    double sx, sy, third;                          // 2/hx, 2/hy, 1/3
    double TT[2][FX_PMAX][FX_PMAX], cN[FX_PMAX], cP[FX_PMAX], L[FX_PMAX], R[FX_PMAX];   // centred flux; [1]: first cell of a Dirichlet line
};

#define DB_CHAIN(acc, COEF, VAL)                         \
    {                                                    \
        acc = __dmul_rn(COEF(0), VAL(0));                \
        _Pragma("unroll") for (int m_ = 1; m_ < P; ++m_) \
            acc = __fma_rn(COEF(m_), VAL(m_), acc);      \
    }
#define DBL(m) g.L[m]
#define DBR(m) g.R[m]

// derivative value at node k of a line from the line's P values and the two neighbour traces
template <int P>
__device__ __forceinline__ double db_out(const DbParams& g, int k, bool first, double s, const double (&u)[P], double tRp, double tLn) {
    double a;
#define CT(m) (first ? g.TT[1][k][m] : g.TT[0][k][m])
#define UU(m) u[m]
    DB_CHAIN(a, CT, UU)
#undef CT
#undef UU
    a = __fma_rn(g.cP[k], tRp, a);
    a = __fma_rn(g.cN[k], tLn, a);
    return __dmul_rn(s, a);
}
// fx_pointwise_dot2(alpha = 1/3, x1, y1, beta = -1/3, x2, y2, gamma = 0): a = RN(alpha x1); b = RN(beta x2); z = fma(a, y1, RN(b y2))
__device__ __forceinline__ double db_pd2(double third, double x1, double y1, double x2, double y2) {
    return __fma_rn(__dmul_rn(third, x1), y1, __dmul_rn(__dmul_rn(-third, x2), y2));
}

// One CTA: tile `tx` of the cell columns, cell rows [j0, j1) (geometry, ring and schedule as dgt_tile: sequence q = cell row
// j0 - 1 + q, iteration it waits for q = it+1, runs the x-phase of row j0+it and the y-phase of row j0-1+it, one barrier).
// STAGE 0: streams f, g -> o0 = out, o1 = h1, o2 = h2.   STAGE 1: streams h1, h2, out -> o0 = out.
template <int P, int NBX, int NS, int STAGE>
__device__ __forceinline__ void dgb_tile(const DbParams& g, const DgtTile& t, const CUtensorMap* const (&mm)[3], const CUtensorMap* const (&mh)[3],
                                         double* __restrict__ o0, double* __restrict__ o1, double* __restrict__ o2,
                                         unsigned long long* bars, int tx, int seg) {
    constexpr int NSTR = STAGE == 0 ? 2 : 3;
    typedef DgtGeom<P, NBX, NSTR, NS> G;
    constexpr int NW = NBX * P;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int Nx = g.Nx, Ny = g.Ny, pitch = Nx * P;
    const int txc = t.wb * NBX, i0 = tx * txc;
    const int j0 = seg * t.rows_per_seg;
    const int j1 = (j0 + t.rows_per_seg < Ny) ? j0 + t.rows_per_seg : Ny;
    const int n = j1 - j0;
    const bool wallx = g.bcx == 1, wally = g.bcy == 1;
    const bool has_pro = !(j0 == 0 && wally), has_top = !(j1 == Ny && wally);
    extern __shared__ __align__(128) double dgt_smem[];
    double2* const hbuf = reinterpret_cast<double2*>(dgt_smem + (size_t)NS * G::STG_D);   // hand-off double2[2][P][SW] (stage B uses .x)
    const unsigned sbase = fx_smem_addr(dgt_smem), full0 = fx_smem_addr(bars);
    constexpr int HBUF = P * G::HSW;                               // (padded cell pitch for P = 4: DgtGeom::HP)
    const int cR = (i0 + txc < Nx) ? i0 + txc : Nx;
    const bool wrapL = i0 == 0 && !wallx, wrapR = cR >= Nx && !wallx;

    // x-phase identity
    const int xb = warp % NBX, xl = warp / NBX;
    const int ci = i0 - 1 + t.wb * xb + lane;
    const bool outside = ci < 0 || ci >= Nx;
    const bool xghost = outside && (wallx || ci < -1 || ci > Nx);
    const bool produce = lane >= 1 && lane <= t.wb && ci < Nx;
    const bool firstx = wallx && ci == 0;
    int xa, hw;
    {
        int cl = ci - i0;
        if (cl < -1 || cl > G::TXM) cl = 0;
        xa = xl * G::BW + G::HE + (cl + 1) * P;
        if (wrapL && ci == -1) xa = G::MAIN_D + xl * G::HW + G::HE;
        if (wrapR && ci == Nx) xa = G::MAIN_D + G::WRAP_D + xl * G::HW;
        if (cl < 0 || cl >= G::TXM) cl = 0;
        hw = xl * G::HSW + cl * G::HP;
    }
    // y-phase identity
    const int ycol = tid < G::SW ? tid : G::SW - 1;
    const bool yact = tid < txc * P && (long long)i0 * P + tid < pitch;
    const int hcol = (ycol / P) * G::HP + ycol % P;                  // this column in a hand-off row
    const int ya = G::HE + P + ycol;
    const long long prow = (long long)pitch;
    const long long obase = (long long)j0 * P * pitch + (long long)i0 * P + tid;
    double* p0 = o0 + obase;
    double* p1 = STAGE == 0 ? o1 + obase : nullptr;
    double* p2 = STAGE == 0 ? o2 + obase : nullptr;

    // producer (the warps take turns)
    const int colM = (i0 - 1) * P - G::HE;
    auto present = [&](int q) { return q == 0 ? has_pro : q == n + 1 ? has_top : true; };
    auto issue = [&](int q) {
        int r = j0 - 1 + q;
        if (r < 0) r += Ny;
        if (r >= Ny) r -= Ny;
        r *= P;
        const unsigned bar = full0 + 8u * (q % NS);
        if (!present(q)) { fx_mbar_arrive(bar); return; }
        const unsigned dst = sbase + (unsigned)(q % NS) * (unsigned)(G::STG_D * 8);
        fx_mbar_expect_tx(bar, (unsigned)NSTR * (G::MAIN_BYTES + (wrapL ? G::WRAP_BYTES : 0u) + (wrapR ? G::WRAP_BYTES : 0u)));
#pragma unroll
        for (int sidx = 0; sidx < NSTR; ++sidx) {
            const unsigned d = dst + (unsigned)(sidx * G::STR_D * 8);
            fx_tma_load_2d(d, mm[sidx], colM, r, bar);
            if (wrapL) fx_tma_load_2d(d + G::MAIN_D * 8, mh[sidx], (Nx - 1) * P - G::HE, r, bar);
            if (wrapR) fx_tma_load_2d(d + (G::MAIN_D + G::WRAP_D) * 8, mh[sidx], 0, r, bar);
        }
    };
    if (tid == 0) {
#pragma unroll 1
        for (int q = 0; q < NS && q <= n + 1; ++q) issue(q);
    }
    int next = NS, pw = 0;

    // the carried column: values of the current cell row (read) and of the next one (loaded now); stage A carries f and g, stage B
    // h2 and out; tRa / tRb: the right (top) traces of the row below
    double ac[P], bc_[P], an[P], bn[P];
    double tRa = 0.0, tRb = 0.0;
#pragma unroll
    for (int l = 0; l < P; ++l) { an[l] = 0.0; bn[l] = 0.0; }
    constexpr int SB = STAGE == 0 ? 1 : 2;                           // second carried stream: g (stage A) / out (stage B)
    constexpr int SA = STAGE == 0 ? 0 : 1;                           // first carried stream: f (stage A) / h2 (stage B)
    if (has_pro) {
        fx_mbar_wait(full0, 0u);
#pragma unroll
        for (int l = 0; l < P; ++l) { an[l] = dgt_smem[SA * G::STR_D + ya + l * G::BW]; bn[l] = dgt_smem[SB * G::STR_D + ya + l * G::BW]; }
    }
#pragma unroll 1
    for (int it = 0; it <= n; ++it) {
        const int q = it + 1;
        const bool have = present(q);
        const double* const sq = dgt_smem + (q % NS) * G::STG_D;
        if (have) fx_mbar_wait(full0 + 8u * (q % NS), (unsigned)((q / NS) & 1));

        // ---- x-phase of cell row j0 + it: centred x derivatives of the line (stage A: of f and g; stage B: of h1) -------------
        if (it < n) {
            double u[P], v[P], tLu, tRu, tLv = 0.0, tRv = 0.0;
#pragma unroll
            for (int m = 0; m < P; ++m) { u[m] = sq[xa + m]; v[m] = STAGE == 0 ? sq[G::STR_D + xa + m] : 0.0; }
#define UU(m) u[m]
#define VV(m) v[m]
            DB_CHAIN(tLu, DBL, UU)
            DB_CHAIN(tRu, DBR, UU)
            if (STAGE == 0) { DB_CHAIN(tLv, DBL, VV) DB_CHAIN(tRv, DBR, VV) }
#undef UU
#undef VV
            if (xghost) { tLu = 0.0; tRu = 0.0; tLv = 0.0; tRv = 0.0; }
            const double tLnu = __shfl_down_sync(0xffffffffu, tLu, 1), tRpu = __shfl_up_sync(0xffffffffu, tRu, 1);
            double tLnv = 0.0, tRpv = 0.0;
            if (STAGE == 0) { tLnv = __shfl_down_sync(0xffffffffu, tLv, 1); tRpv = __shfl_up_sync(0xffffffffu, tRv, 1); }
            if (produce) {
                double2* const h = hbuf + (it & 1) * HBUF + hw;
#pragma unroll
                for (int k = 0; k < P; ++k)
                    h[k] = make_double2(db_out<P>(g, k, firstx, g.sx, u, tRpu, tLnu), STAGE == 0 ? db_out<P>(g, k, firstx, g.sx, v, tRpv, tLnv) : 0.0);
            }
        }

        // ---- y-phase of cell row r = j0 - 1 + it ----------------------------------------------------------------------------------
#pragma unroll
        for (int l = 0; l < P; ++l) { ac[l] = an[l]; bc_[l] = bn[l]; }
        if (have) {
#pragma unroll
            for (int l = 0; l < P; ++l) { an[l] = sq[SA * G::STR_D + ya + l * G::BW]; bn[l] = sq[SB * G::STR_D + ya + l * G::BW]; }
        }
        double tLna, tLnb = 0.0, tRac, tRbc = 0.0;
#define AN(m) an[m]
#define BN(m) bn[m]
#define AC(m) ac[m]
#define BC(m) bc_[m]
        DB_CHAIN(tLna, DBL, AN)
        DB_CHAIN(tRac, DBR, AC)
        if (STAGE == 0) { DB_CHAIN(tLnb, DBL, BN) DB_CHAIN(tRbc, DBR, BC) }
#undef AN
#undef BN
#undef AC
#undef BC
        if (!have) { tLna = 0.0; tLnb = 0.0; }                          // beyond a wall: zero ghost trace
        if (it == 0) {
            if (!has_pro) { tRac = 0.0; tRbc = 0.0; }                    // (the segment starts at a wall: no row below)
        } else {
            const int r = j0 - 1 + it;
            const bool firsty = wally && r == 0;
            const double2* const h = hbuf + ((it - 1) & 1) * HBUF + hcol;
            double w0[P], w1[P], w2[P];
#pragma unroll
            for (int l = 0; l < P; ++l) {
                const double2 hx = h[l * G::HSW];
                const double ay = db_out<P>(g, l, firsty, g.sy, ac, tRa, tLna);
                if (STAGE == 0) {
                    const double by = db_out<P>(g, l, firsty, g.sy, bc_, tRb, tLnb);
                    // f = ac, g = bc_, f_x = hx.x, g_x = hx.y, f_y = ay, g_y = by
                    w0[l] = db_pd2(g.third, hx.x, by, ay, hx.y);         // 1/3 (f_x g_y - f_y g_x)
                    w1[l] = db_pd2(g.third, ac[l], by, bc_[l], ay);      // 1/3 (f g_y - g f_y)
                    w2[l] = db_pd2(g.third, bc_[l], hx.x, ac[l], hx.y);  // 1/3 (g f_x - f g_x)
                } else {
                    // out <- fma(1, D_x h1, RN(1 * out)); out <- fma(1, D_y h2, RN(1 * out))
                    const double s1 = __fma_rn(1.0, hx.x, __dmul_rn(1.0, bc_[l]));
                    w0[l] = __fma_rn(1.0, ay, __dmul_rn(1.0, s1));
                }
            }
            if (yact) {
#pragma unroll
                for (int l = 0; l < P; ++l) {
                    p0[l * prow] = w0[l];
                    if (STAGE == 0) { p1[l * prow] = w1[l]; p2[l * prow] = w2[l]; }
                }
            }
            p0 += P * prow;
            if (STAGE == 0) { p1 += P * prow; p2 += P * prow; }
        }
        tRa = tRac; tRb = tRbc;
        __syncthreads();
        const int lim = (it + 1 + NS < n + 1) ? it + 1 + NS : n + 1;
        if (warp == pw && lane == 0)
            for (int qq = next; qq <= lim; ++qq) issue(qq);
        if (lim >= next) next = lim + 1;
        pw = (pw + 1 == NW) ? 0 : pw + 1;
    }
}

#undef DBL
#undef DBR
#endif
