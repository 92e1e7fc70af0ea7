// oracle/fxo.cpp  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU oracle for the hot path of arXiv:1807.01971 (Feltor):
// exactly rounded dot product, axpby, pointwise_dot, the 2-D dG elliptic operator and the
// preconditioned CG built from them.  It exists to define what the CUDA library (libfx.so) must
// compute.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load it.  It shares no code, header, table or technique with the CUDA path:
//   * the dot is the DEFINITION  RN(sum_i x_i*y_i)  evaluated with a big integer (no TwoSum /
//     TwoProd / floating-point expansion anywhere in this file);
//   * the dG operator exists twice: as explicit block matrices applied in 113-bit arithmetic (the
//     definition) and as the canonical fp64 operation sequence (DESIGN.md
//     section 3.4) that fixes "type and order of execution of floating point operations" as the paper
//     prescribes for every non-reduction primitive (section 3.2).
// Citations "P:n" are PAPER.md line numbers.  Readings of silent points are DESIGN.md "Qn".
//
// Pins (tests/test_oracle_*.py, all CPU): rational brute force, the paper's associativity example
// (P:158), closed forms, permutation/scaling invariances, Fig. 2's integral, GL closed
// forms and identities, symmetry / SPD / polynomial exactness / P=1 five-point stencil / convergence
// order of the operator, dense direct solve for CG.
// Parity unpinned: equality with Feltor's own discretisation and stopping rule (its source is not
// available here; Q8) -- only the properties above are claimed.
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared fxo.cpp -o liboracle.so -lquadmath

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

typedef __float128 q128;
typedef unsigned __int128 u128;

// ------------------------------------------------------------------------------------------------
// 1. Exact dot product: RN( sum_i x_i * y_i ), sum and products over the reals.
//    P:9 "exactly rounded dot product"; "correctly rounded (rounding-to-nearest)";
//    P:172 long accumulator = scaled integer over the whole exponent range (Kulisch: 4288 bit).
//    DESIGN.md Q1-Q6.
// ------------------------------------------------------------------------------------------------

static const int NLIMB = 68;        // 68 x 64 = 4352 bit, limb k weighs 2^(64k - 2176)
static const int BIAS_BITS = 2176;  // bit b of the integer weighs 2^(b - 2176)

struct BigAcc {
    uint64_t limb[NLIMB];           // two's complement
    int nan_flag, pinf_flag, ninf_flag;
};

static void acc_clear(BigAcc& a) { std::memset(&a, 0, sizeof(a)); }

// add (sub==0) or subtract (sub==1) the 3-limb magnitude w[0..2] at limb position q
static void acc_addsub(BigAcc& a, int q, const uint64_t w[3], int sub) {
    if (!sub) {
        unsigned carry = 0;
        for (int k = q; k < NLIMB; ++k) {
            uint64_t add = (k - q < 3) ? w[k - q] : 0;
            if (k - q >= 3 && !carry) break;
            u128 s = (u128)a.limb[k] + add + carry;
            a.limb[k] = (uint64_t)s;
            carry = (unsigned)(s >> 64);
        }
    } else {
        unsigned borrow = 0;
        for (int k = q; k < NLIMB; ++k) {
            uint64_t subv = (k - q < 3) ? w[k - q] : 0;
            if (k - q >= 3 && !borrow) break;
            u128 d = (u128)a.limb[k] - subv - borrow;
            a.limb[k] = (uint64_t)d;
            borrow = (unsigned)((d >> 64) & 1);
        }
    }
}

// DESIGN.md 3.1 steps 1-3 and 5: decode, exact product, accumulate; non-finite -> flags
static void acc_add_product(BigAcc& a, double x, double y) {
    uint64_t bx, by;
    std::memcpy(&bx, &x, 8);
    std::memcpy(&by, &y, 8);
    int sx = (int)(bx >> 63), sy = (int)(by >> 63);
    int ex = (int)((bx >> 52) & 0x7ff), ey = (int)((by >> 52) & 0x7ff);
    uint64_t fx = bx & 0xfffffffffffffULL, fy = by & 0xfffffffffffffULL;
    bool x_nan = (ex == 0x7ff && fx != 0), y_nan = (ey == 0x7ff && fy != 0);
    bool x_inf = (ex == 0x7ff && fx == 0), y_inf = (ey == 0x7ff && fy == 0);
    bool x_zero = (ex == 0 && fx == 0), y_zero = (ey == 0 && fy == 0);
    if (x_nan || y_nan) { a.nan_flag = 1; return; }
    if (x_inf || y_inf) {
        if (x_zero || y_zero) { a.nan_flag = 1; return; }   // 0 * inf
        if (sx ^ sy) a.ninf_flag = 1; else a.pinf_flag = 1;
        return;
    }
    uint64_t Mx = ex ? (fx | (1ULL << 52)) : fx;             // hidden bit iff biased exponent > 0
    uint64_t My = ey ? (fy | (1ULL << 52)) : fy;
    int Ex = (ex ? ex : 1) - 1075, Ey = (ey ? ey : 1) - 1075; // value = (-1)^s * M * 2^E
    u128 m = (u128)Mx * My;                                   // < 2^106, exact
    if (m == 0) return;
    int pos = Ex + Ey + BIAS_BITS;                            // in [28, 4118]
    int q = pos / 64, s = pos % 64;
    uint64_t w[3];
    uint64_t mlo = (uint64_t)m, mhi = (uint64_t)(m >> 64);
    if (s == 0) { w[0] = mlo; w[1] = mhi; w[2] = 0; }
    else { w[0] = mlo << s; w[1] = (mhi << s) | (mlo >> (64 - s)); w[2] = mhi >> (64 - s); }
    acc_addsub(a, q, w, sx ^ sy);
}

static int big_bit(const uint64_t* mag, int b) { return b < 0 ? 0 : (int)((mag[b / 64] >> (b % 64)) & 1); }

// DESIGN.md 3.1 step 4: one rounding to nearest, ties to even, gradual underflow, overflow -> inf
static double acc_round(const BigAcc& a) {
    if (a.nan_flag || (a.pinf_flag && a.ninf_flag)) {
        uint64_t qnan = 0x7FF8000000000000ULL; double r; std::memcpy(&r, &qnan, 8); return r;
    }
    if (a.pinf_flag) return HUGE_VAL;
    if (a.ninf_flag) return -HUGE_VAL;
    uint64_t mag[NLIMB];
    int neg = (int)(a.limb[NLIMB - 1] >> 63);
    if (neg) {                                   // magnitude = two's complement negation
        unsigned carry = 1;
        for (int k = 0; k < NLIMB; ++k) { u128 s = (u128)(~a.limb[k]) + carry; mag[k] = (uint64_t)s; carry = (unsigned)(s >> 64); }
    } else std::memcpy(mag, a.limb, sizeof(mag));
    int t = -1;
    for (int k = NLIMB - 1; k >= 0 && t < 0; --k)
        if (mag[k]) for (int b = 63; b >= 0; --b) if ((mag[k] >> b) & 1) { t = 64 * k + b; break; }
    if (t < 0) return 0.0;                       // exact zero -> +0.0 (Q3)
    int p = t - 52;                              // lsb kept
    const int PMIN = -1074 + BIAS_BITS;          // lsb of the subnormal grid
    if (p < PMIN) p = PMIN;
    uint64_t mant = 0;
    for (int b = p + 52; b >= p; --b) mant = (mant << 1) | (uint64_t)big_bit(mag, b);
    int round_bit = big_bit(mag, p - 1);
    int sticky = 0;
    for (int b = p - 2; b >= 0 && !sticky; --b) sticky |= big_bit(mag, b);
    if (round_bit && (sticky || (mant & 1))) mant += 1;       // ties to even
    double r = std::ldexp((double)mant, p - BIAS_BITS);       // exact, or +inf on overflow
    return neg ? -r : r;
}

extern "C" double fxo_exdot(const double* x, const double* y, int64_t n) {
    BigAcc a; acc_clear(a);
    for (int64_t i = 0; i < n; ++i) acc_add_product(a, x[i], y[i]);
    return acc_round(a);
}

// the 68-limb two's complement accumulator itself (+ the three non-finite flags)
extern "C" double fxo_exdot_digits(const double* x, const double* y, int64_t n, uint64_t limbs[68], int32_t flags[3]) {
    BigAcc a; acc_clear(a);
    for (int64_t i = 0; i < n; ++i) acc_add_product(a, x[i], y[i]);
    std::memcpy(limbs, a.limb, sizeof(a.limb));
    if (flags) { flags[0] = a.nan_flag; flags[1] = a.pinf_flag; flags[2] = a.ninf_flag; }
    return acc_round(a);
}

// Weighted dot sum_i x_i w_i y_i ("we also provide a function computing the weighted sum", rounding of the triple
// product not specified): reading Q14 -- u_i = RN(x_i * w_i) in fp64, then the exact dot of u and y.  w == 1 reduces it
// to the exact dot.  Exact sum: the exact dot with ones (EXSUM).
extern "C" double fxo_exdot3(const double* x, const double* w, const double* y, int64_t n) {
    BigAcc a; acc_clear(a);
    for (int64_t i = 0; i < n; ++i) { volatile double u = x[i] * w[i]; acc_add_product(a, u, y[i]); }
    return acc_round(a);
}
extern "C" double fxo_exsum(const double* x, int64_t n) {
    BigAcc a; acc_clear(a);
    for (int64_t i = 0; i < n; ++i) acc_add_product(a, x[i], 1.0);
    return acc_round(a);
}

// Single-precision inputs, exact accumulation (an exact dot lets single precision keep its accuracy):
// RN_double( sum_i x_i * y_i ) for binary32 x, y -- every product is formed exactly (48-bit mantissa) as in fxo_exdot.
extern "C" double fxo_exdot_f32(const float* x, const float* y, int64_t n) {
    BigAcc a; acc_clear(a);
    for (int64_t i = 0; i < n; ++i) acc_add_product(a, (double)x[i], (double)y[i]);
    return acc_round(a);
}

// Running correctly rounded sums with feedback -- the input construction of BASELINE.json config 1, "Family B" (SURVEY
// 8d: "the other half are constructed to cancel so the exact sum is tiny").  For j = start .. n-1, in this order:
//   sigma_j = RN( sum_{i<j} x_i*y_i )   (the definition above, one rounding);   y_j = RN( RN(t_j - sigma_j) / x_j ),
// so that after element j the exact running sum is t_j up to rounding residues.  x, t: inputs; y[start..n) is written.
// Pin: tests/test_oracle_exdot.py recomputes every sigma_j with fractions.Fraction.
extern "C" void fxo_exdot_cancel_fill(const double* x, double* y, int64_t start, int64_t n, const double* t) {
    BigAcc a; acc_clear(a);
    for (int64_t i = 0; i < start; ++i) acc_add_product(a, x[i], y[i]);
    for (int64_t j = start; j < n; ++j) {
        const double sigma = acc_round(a);
        volatile double d = t[j] - sigma;
        volatile double q = d / x[j];
        y[j] = q;
        acc_add_product(a, x[j], y[j]);
    }
}

// round an externally supplied accumulator (used by the "concatenation = integer sum" pin)
extern "C" double fxo_round_digits(const uint64_t limbs[68]) {
    BigAcc a; acc_clear(a); std::memcpy(a.limb, limbs, sizeof(a.limb));
    return acc_round(a);
}

// ------------------------------------------------------------------------------------------------
// 2. Vector primitives in canonical order (fix type and order of operations, explicit
//    FMA, two roundings instead of three).  DESIGN.md 3.2 / Q13.
// ------------------------------------------------------------------------------------------------

extern "C" void fxo_axpby(double alpha, const double* x, double beta, double* y, int64_t n) {
    if (beta == 0.0) { for (int64_t i = 0; i < n; ++i) y[i] = alpha * x[i]; return; }
    for (int64_t i = 0; i < n; ++i) { double t = beta * y[i]; y[i] = std::fma(alpha, x[i], t); }
}

extern "C" void fxo_pointwise_dot(double alpha, const double* x1, const double* x2, double beta, double* y, int64_t n) {
    if (beta == 0.0) { for (int64_t i = 0; i < n; ++i) { double u = alpha * x1[i]; y[i] = u * x2[i]; } return; }
    for (int64_t i = 0; i < n; ++i) { double u = alpha * x1[i]; double t = beta * y[i]; y[i] = std::fma(u, x2[i], t); }
}

// ------------------------------------------------------------------------------------------------
// 3. Gauss-Legendre reference element in 113-bit arithmetic (Fig. 2: grid of P
//    Gauss-Legendre nodes per cell and direction; P = number of polynomial coefficients).
//    DESIGN.md 3.3.
// ------------------------------------------------------------------------------------------------

static const int PMAX = 5;

struct RefElem {
    int P;
    q128 xi[PMAX], w[PMAX];          // nodes ascending, weights
    q128 D[PMAX][PMAX];              // D[k][m] = l_m'(xi_k)
    q128 L[PMAX], R[PMAX];           // l_m(-1), l_m(+1)
};

static void legendre(int n, q128 x, q128& pn, q128& pnm1) {   // three-term recurrence
    q128 p0 = 1, p1 = x;
    if (n == 0) { pn = 1; pnm1 = 0; return; }
    for (int k = 2; k <= n; ++k) { q128 p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k; p0 = p1; p1 = p2; }
    pn = p1; pnm1 = p0;
}

static void ref_elem(int P, RefElem& e) {
    e.P = P;
    const q128 pi = 3.14159265358979323846264338327950288419716939937510Q;
    for (int k = 0; k < P / 2; ++k) {          // the negative roots of P_P by Newton, ascending
        q128 x = -(q128)std::cos((double)(pi * (k + 0.75Q) / (P + 0.5Q)));
        for (int it = 0; it < 100; ++it) {
            q128 pn, pm; legendre(P, x, pn, pm);
            q128 dp = P * (x * pn - pm) / (x * x - 1);      // P_P'(x)
            x -= pn / dp;
        }
        e.xi[k] = x;
    }
    if (P % 2 == 1) e.xi[P / 2] = 0;                                   // middle root is exactly 0
    for (int k = (P + 1) / 2; k < P; ++k) e.xi[k] = -e.xi[P - 1 - k];  // xi_k = -xi_{P-1-k}
    for (int k = 0; k < P; ++k) {
        q128 pn, pm; legendre(P, e.xi[k], pn, pm);
        q128 x = e.xi[k];
        q128 dp = (P == 1) ? 1 : P * (x * pn - pm) / (x * x - 1);
        e.w[k] = 2 / ((1 - x * x) * dp * dp);
    }
    for (int m = 0; m < P; ++m) {              // Lagrange basis on the nodes
        q128 l = 1, r = 1;
        for (int j = 0; j < P; ++j) if (j != m) { l *= (-1 - e.xi[j]) / (e.xi[m] - e.xi[j]); r *= (1 - e.xi[j]) / (e.xi[m] - e.xi[j]); }
        e.L[m] = l; e.R[m] = r;
    }
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) {
        if (k == m) {                           // l_k'(xi_k) = sum_{j!=k} 1/(xi_k - xi_j)
            q128 s = 0;
            for (int j = 0; j < P; ++j) if (j != k) s += 1 / (e.xi[k] - e.xi[j]);
            if (P % 2 == 1 && k == P / 2) s = 0; // antisymmetric sum, exactly 0
            e.D[k][m] = s;
        } else {                                // l_m'(xi_k) = prod_{j!=m,k}(xi_k-xi_j) / prod_{j!=m}(xi_m-xi_j)
            q128 num = 1, den = 1;
            for (int j = 0; j < P; ++j) { if (j != m && j != k) num *= (e.xi[k] - e.xi[j]); if (j != m) den *= (e.xi[m] - e.xi[j]); }
            e.D[k][m] = num / den;
        }
    }
}

// fp64 tables, each entry rounded once from the 113-bit value (DESIGN.md 3.4 "Tables")
struct Tables {
    int P;
    double xi[PMAX], w[PMAX], L[PMAX], R[PMAX], B[PMAX];
    double T0[PMAX][PMAX], T0L[PMAX][PMAX], WW[PMAX][PMAX], D[PMAX][PMAX];
};

static double snap(q128 v) { q128 a = v < 0 ? -v : v; return a < 1e-28Q ? 0.0 : (double)v; }

static void make_tables(int P, Tables& t) {
    RefElem e; ref_elem(P, e);
    t.P = P;
    for (int k = 0; k < P; ++k) {
        t.xi[k] = snap(e.xi[k]); t.w[k] = (double)e.w[k]; t.L[k] = snap(e.L[k]); t.R[k] = snap(e.R[k]);
        t.B[k] = snap(e.R[k] / e.w[k]);
        for (int m = 0; m < P; ++m) {
            q128 t0 = e.D[k][m] - e.R[k] * e.R[m] / e.w[k];
            t.T0[k][m] = snap(t0);
            t.T0L[k][m] = snap(t0 + e.L[k] * e.L[m] / e.w[k]);
            t.WW[k][m] = (double)(e.w[k] * e.w[m]);
            t.D[k][m] = snap(e.D[k][m]);
        }
    }
}

// out: xi[P], w[P], L[P], R[P], B[P], then T0, T0L, WW, D (each P*P row-major)
extern "C" int fxo_dg_tables(int32_t P, double* out) {
    if (P < 1 || P > PMAX) return -1;
    Tables t; make_tables(P, t);
    double* o = out;
    for (int k = 0; k < P; ++k) *o++ = t.xi[k];
    for (int k = 0; k < P; ++k) *o++ = t.w[k];
    for (int k = 0; k < P; ++k) *o++ = t.L[k];
    for (int k = 0; k < P; ++k) *o++ = t.R[k];
    for (int k = 0; k < P; ++k) *o++ = t.B[k];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.T0[k][m];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.T0L[k][m];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.WW[k][m];
    for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = t.D[k][m];
    return 0;
}

// ------------------------------------------------------------------------------------------------
// 4. Grid, weights.  Fig. 2: CartesianGrid2d(x0,x1,y0,y1,P,Nx,Ny), volume form.
//    Layout (Q15): row-major (Ny*P) x (Nx*P) image, x fastest:
//        idx = ((j*P + l)*Nx + i)*P + k     cell (i,j), node (k,l)
// ------------------------------------------------------------------------------------------------

struct fxo_grid { int32_t Nx, Ny, P; double lx, ly; int32_t bcx, bcy; };
// bc of one direction: 0 = PER, 1 = DIR (both walls), 2 = NEU (both walls), 3 = DIR_NEU (Dirichlet at the lower wall,
// Neumann at the upper one), 4 = NEU_DIR.  NEU and the mixed kinds: SURVEY 8f-4, reading DESIGN.md Q23.
enum { BC_PER = 0, BC_DIR = 1, BC_NEU = 2, BC_DIR_NEU = 3, BC_NEU_DIR = 4 };
static int wall_lo(int bc) { return bc == BC_PER ? BC_PER : (bc == BC_DIR || bc == BC_DIR_NEU) ? BC_DIR : BC_NEU; }
static int wall_hi(int bc) { return bc == BC_PER ? BC_PER : (bc == BC_DIR || bc == BC_NEU_DIR) ? BC_DIR : BC_NEU; }
static bool bc_ok(int bc, int N) { return bc >= BC_PER && bc <= BC_NEU_DIR && !(bc == BC_DIR_NEU && N < 2); }

static int grid_ok(const fxo_grid* g) {
    return g && g->Nx >= 1 && g->Ny >= 1 && g->P >= 1 && g->P <= PMAX && g->lx > 0 && g->ly > 0 &&
           bc_ok(g->bcx, g->Nx) && bc_ok(g->bcy, g->Ny);
}

// the stand-alone derivatives and the bracket are defined for PER and DIR only (Q21, Q23)
static bool deriv_bc_ok(const fxo_grid* g) { return g->bcx <= BC_DIR && g->bcy <= BC_DIR; }

static inline int64_t gidx(const fxo_grid* g, int i, int j, int k, int l) {
    return (((int64_t)j * g->P + l) * g->Nx + i) * g->P + k;
}

// W[idx] = RN( RN(RN(hx*hy)/4) * WW[l][k] ),  V[idx] = RN(1/W[idx])
extern "C" int fxo_dg_weights(const fxo_grid* g, double* W, double* V) {
    if (!grid_ok(g)) return -1;
    Tables t; make_tables(g->P, t);
    double hx = g->lx / g->Nx, hy = g->ly / g->Ny;
    double a = (hx * hy) / 4;
    for (int j = 0; j < g->Ny; ++j) for (int l = 0; l < g->P; ++l)
        for (int i = 0; i < g->Nx; ++i) for (int k = 0; k < g->P; ++k) {
            double w = a * t.WW[l][k];
            int64_t id = gidx(g, i, j, k, l);
            if (W) W[id] = w;
            if (V) V[id] = 1.0 / w;
        }
    return 0;
}

// node coordinates x(i,k) = hx*(i + (1+xi_k)/2) (for tests that evaluate functions on the grid)
extern "C" int fxo_dg_nodes(const fxo_grid* g, double* xs, double* ys) {
    if (!grid_ok(g)) return -1;
    RefElem e; ref_elem(g->P, e);
    q128 hx = (q128)g->lx / g->Nx, hy = (q128)g->ly / g->Ny;
    for (int i = 0; i < g->Nx; ++i) for (int k = 0; k < g->P; ++k) xs[i * g->P + k] = (double)(hx * (i + (1 + e.xi[k]) / 2));
    for (int j = 0; j < g->Ny; ++j) for (int l = 0; l < g->P; ++l) ys[j * g->P + l] = (double)(hy * (j + (1 + e.xi[l]) / 2));
    return 0;
}

// ------------------------------------------------------------------------------------------------
// 5. dG elliptic operator, DEFINITION: explicit 1-D block matrices, 113-bit arithmetic.
//    The paper names the construction only by reference (dG derivatives [21], elliptic
//    discretisation after [12],[6]); the reading is DESIGN.md 3.3 / Q8:
//      F(N,h,bc): forward-flux derivative.  block row n:
//          F[n][n]   = (2/h) (D - W^-1 R R^T)            (+ (2/h) W^-1 L L^T  if n==0 and the lower wall is DIR)
//          F[n][n+1] = (2/h)  W^-1 R L^T                 (PER: n+1 mod N;  walls: absent for n==N-1)
//      J(N,bc): jump  sum_faces [v][u], un-normed.  block row n:
//          J[n][n] = R R^T + L L^T,  J[n][n+1] = -R L^T,  J[n][n-1] = -L R^T   (PER wraps; walls: absent)
//      Neumann wall (Q23): the ghost cell mirrors the interior trace, so the face carries neither a jump nor a
//      flux correction: at an upper NEU wall F[N-1][N-1] = (2/h) D (the -W^-1 R R^T term cancels against the
//      mirrored neighbour) and J[N-1][N-1] = L L^T; at a lower NEU wall F[0][0] is the interior block (the forward
//      flux takes the cell's own value there anyway) and J[0][0] = R R^T.
//      S = Fx^T diag(W chi) Fx + Fy^T diag(W chi) Fy + diag(Wy) (x) Jx + Jy (x) diag(Wx),  A = diag(V) S.
// ------------------------------------------------------------------------------------------------

// dense (N*P) x (N*P) matrices, row-major, in q128
static void build_F(const RefElem& e, int N, q128 h, int bc, std::vector<q128>& F) {
    int P = e.P, n = N * P;
    F.assign((size_t)n * n, 0);
    q128 s = 2 / h;
    for (int c = 0; c < N; ++c) for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) {
        q128 d = e.D[k][m];
        if (!(c == N - 1 && wall_hi(bc) == BC_NEU)) d -= e.R[k] * e.R[m] / e.w[k];
        if (c == 0 && wall_lo(bc) == BC_DIR) d += e.L[k] * e.L[m] / e.w[k];
        F[(size_t)(c * P + k) * n + (c * P + m)] += s * d;
        int cn = c + 1;
        if (cn == N) { if (bc == BC_PER) cn = 0; else continue; }
        F[(size_t)(c * P + k) * n + (cn * P + m)] += s * e.R[k] * e.L[m] / e.w[k];
    }
}

static void build_J(const RefElem& e, int N, int bc, std::vector<q128>& J) {
    int P = e.P, n = N * P;
    J.assign((size_t)n * n, 0);
    for (int c = 0; c < N; ++c) for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) {
        if (!(c == N - 1 && wall_hi(bc) == BC_NEU)) J[(size_t)(c * P + k) * n + (c * P + m)] += e.R[k] * e.R[m];
        if (!(c == 0 && wall_lo(bc) == BC_NEU)) J[(size_t)(c * P + k) * n + (c * P + m)] += e.L[k] * e.L[m];
        int cn = c + 1, cp = c - 1;
        if (cn == N) cn = (bc == BC_PER) ? 0 : -1;
        if (cp < 0) cp = (bc == BC_PER) ? N - 1 : -1;
        if (cn >= 0) J[(size_t)(c * P + k) * n + (cn * P + m)] += -e.R[k] * e.L[m];
        if (cp >= 0) J[(size_t)(c * P + k) * n + (cp * P + m)] += -e.L[k] * e.R[m];
    }
}

// 1-D matrices rounded to double, for the numpy-side checks (symmetry, exactness on polynomials ...)
extern "C" int fxo_dg_matrix_1d(int32_t N, int32_t P, double h, int32_t bc, double* F_out, double* J_out) {
    if (N < 1 || P < 1 || P > PMAX || !(h > 0)) return -1;
    RefElem e; ref_elem(P, e);
    std::vector<q128> F, J;
    build_F(e, N, (q128)h, bc, F); build_J(e, N, bc, J);
    size_t nn = (size_t)N * P * N * P;
    for (size_t a = 0; a < nn; ++a) { if (F_out) F_out[a] = (double)F[a]; if (J_out) J_out[a] = (double)J[a]; }
    return 0;
}

// y = S x (normed==0) or A x = V o (S x) (normed==1), every product/sum in q128, rounded once at
// the end; scale = (|Fx^T||W chi||Fx| + |Fy^T||W chi||Fy| + |J|)|x| evaluated the same way.
// Dense 1-D matrices: meant for grids up to a few hundred nodes per direction.
// (zfac: 1 for the 2-D operator; the plane weight hz of a 3-D product grid for its symmetric form, section 8 below --
// a factor of exactly 1 changes no bit of the 2-D results)
static int apply_definition_q(const fxo_grid* g, const double* chi, const double* x, int32_t normed, q128 zfac,
                              double* y, double* scale) {
    if (!grid_ok(g)) return -1;
    const int P = g->P, Nx = g->Nx, Ny = g->Ny, nx = Nx * P, ny = Ny * P;
    RefElem e; ref_elem(P, e);
    q128 hx = (q128)g->lx / Nx, hy = (q128)g->ly / Ny;   // lx/Nx in 113 bit: the definition does not round h
    std::vector<q128> Fx, Fy, Jx, Jy;
    build_F(e, Nx, hx, g->bcx, Fx); build_F(e, Ny, hy, g->bcy, Fy);
    build_J(e, Nx, g->bcx, Jx); build_J(e, Ny, g->bcy, Jy);
    auto wx = [&](int c) { return hx / 2 * e.w[c % P]; };   // 1-D weights, c = column (node) index
    auto wy = [&](int r) { return hy / 2 * e.w[r % P]; };
    size_t n = (size_t)nx * ny;
    std::vector<q128> gx(n), gy(n), agx(n), agy(n), out(n, 0), aout(n, 0);
    auto at = [&](int r, int c) { return (size_t)r * nx + c; };
    auto qabs = [](q128 v) { return v < 0 ? -v : v; };
    // gx = W chi (Fx x) along rows; gy = W chi (Fy x) along columns
    for (int r = 0; r < ny; ++r) for (int c = 0; c < nx; ++c) {
        q128 s = 0, a = 0, s2 = 0, a2 = 0;
        for (int m = 0; m < nx; ++m) { q128 f = Fx[(size_t)c * nx + m]; if (f != 0) { s += f * x[at(r, m)]; a += qabs(f) * qabs((q128)x[at(r, m)]); } }
        for (int m = 0; m < ny; ++m) { q128 f = Fy[(size_t)r * ny + m]; if (f != 0) { s2 += f * x[at(m, c)]; a2 += qabs(f) * qabs((q128)x[at(m, c)]); } }
        q128 wc = wx(c) * wy(r) * chi[at(r, c)];
        gx[at(r, c)] = wc * s; agx[at(r, c)] = qabs(wc) * a;
        gy[at(r, c)] = wc * s2; agy[at(r, c)] = qabs(wc) * a2;
    }
    for (int r = 0; r < ny; ++r) for (int c = 0; c < nx; ++c) {
        q128 s = 0, a = 0;
        for (int m = 0; m < nx; ++m) {       // (Fx^T gx)_c = sum_m Fx[m][c] gx_m ;  jump: Wy * Jx
            q128 f = Fx[(size_t)m * nx + c]; if (f != 0) { s += f * gx[at(r, m)]; a += qabs(f) * agx[at(r, m)]; }
            q128 jj = Jx[(size_t)c * nx + m]; if (jj != 0) { s += wy(r) * jj * x[at(r, m)]; a += wy(r) * qabs(jj) * qabs((q128)x[at(r, m)]); }
        }
        for (int m = 0; m < ny; ++m) {
            q128 f = Fy[(size_t)m * ny + r]; if (f != 0) { s += f * gy[at(m, c)]; a += qabs(f) * agy[at(m, c)]; }
            q128 jj = Jy[(size_t)r * ny + m]; if (jj != 0) { s += wx(c) * jj * x[at(m, c)]; a += wx(c) * qabs(jj) * qabs((q128)x[at(m, c)]); }
        }
        out[at(r, c)] = s; aout[at(r, c)] = a;
    }
    for (int r = 0; r < ny; ++r) for (int c = 0; c < nx; ++c) {
        q128 v = (normed ? 1 / (wx(c) * wy(r)) : (q128)1) * zfac;
        if (y) y[at(r, c)] = (double)(v * out[at(r, c)]);
        if (scale) scale[at(r, c)] = (double)(v * aout[at(r, c)]);
    }
    return 0;
}
extern "C" int fxo_dg_apply_definition(const fxo_grid* g, const double* chi, const double* x, int32_t normed,
                                       double* y, double* scale) {
    return apply_definition_q(g, chi, x, normed, (q128)1, y, scale);
}

// ------------------------------------------------------------------------------------------------
// 6. dG elliptic operator, CANONICAL fp64 evaluation order.  Every intermediate has
//    one defining expression; "chain over m" = acc = c[0]*v[0]; acc = fma(c[m], v[m], acc), m=1..P-1.
//    This is the sequence the CUDA kernel must reproduce bit for bit.
// ------------------------------------------------------------------------------------------------

struct Canon {
    Tables t;
    double cxx, cyy, JX[PMAX], JY[PMAX], vol4;
};

static void make_canon(const fxo_grid* g, Canon& c) {
    make_tables(g->P, c.t);
    double hx = g->lx / g->Nx, hy = g->ly / g->Ny;
    c.cxx = hy / hx; c.cyy = hx / hy;
    for (int l = 0; l < g->P; ++l) { c.JX[l] = (hy / 2) * c.t.w[l]; c.JY[l] = (hx / 2) * c.t.w[l]; }   // jf = 1
    c.vol4 = (hx * hy) / 4;
}

// One line of N cells with P nodes each (stride between consecutive values = stride):
//   s_hat[n*P+k], j_hat[n*P+k] from u[], cw[] (cw = RN(WW*chi) along the same line)
static void line_ops(const Tables& t, int N, int bc, const double* u, const double* cw, double* s_hat, double* j_hat) {
    const int P = t.P;
    std::vector<double> tL(N + 2), tR(N + 2), tB(N + 2), f((size_t)N * P);
    // step 1: traces.  index shift +1 so that [0] is the ghost n=-1 and [N+1] the ghost n=N
    for (int n = 0; n < N; ++n) {
        double aL = t.L[0] * u[n * P], aR = t.R[0] * u[n * P];
        for (int m = 1; m < P; ++m) { aL = std::fma(t.L[m], u[n * P + m], aL); aR = std::fma(t.R[m], u[n * P + m], aR); }
        tL[n + 1] = aL; tR[n + 1] = aR;
    }
    if (bc == BC_PER) { tL[N + 1] = tL[1]; tR[0] = tR[N]; tL[0] = tL[N]; tR[N + 1] = tR[1]; }
    else { tL[N + 1] = 0; tR[0] = 0; tL[0] = 0; tR[N + 1] = 0; }
    // cell tables: T0L in the first cell of a line that starts at a DIR wall; D in the last cell of a line that ends
    // at a NEU wall (Q23; with the zero ghost trace above, step 2 then gives the plain in-cell derivative there)
    auto table = [&](int n) -> const double (*)[PMAX] {
        if (n == 0 && wall_lo(bc) == BC_DIR) return t.T0L;
        if (n == N - 1 && wall_hi(bc) == BC_NEU) return t.D;
        return t.T0;
    };
    // steps 2,3: reference gradient, flux, flux trace
    for (int n = 0; n < N; ++n) {
        const double (*T)[PMAX] = table(n);
        double aB = 0;
        for (int k = 0; k < P; ++k) {
            double a = T[k][0] * u[n * P];
            for (int m = 1; m < P; ++m) a = std::fma(T[k][m], u[n * P + m], a);
            double ghat = std::fma(t.B[k], tL[n + 2], a);
            double fl = cw[n * P + k] * ghat;
            f[(size_t)n * P + k] = fl;
            aB = (k == 0) ? t.B[0] * fl : std::fma(t.B[k], fl, aB);
        }
        tB[n + 1] = aB;
    }
    tB[0] = (bc == BC_PER) ? tB[N] : 0;
    // steps 4,5: adjoint and jump
    for (int n = 0; n < N; ++n) {
        const double (*T)[PMAX] = table(n);
        // the jump's ghost at a NEU wall is the mirror image of the cell's own trace: the difference is +0
        double gR = (n == 0 && wall_lo(bc) == BC_NEU) ? tL[1] : tR[n];
        double gL = (n == N - 1 && wall_hi(bc) == BC_NEU) ? tR[N] : tL[n + 2];
        double dl = tL[n + 1] - gR;             // own left trace - left neighbour's right trace
        double dr = tR[n + 1] - gL;             // own right trace - right neighbour's left trace
        for (int k = 0; k < P; ++k) {
            double a = T[0][k] * f[(size_t)n * P];
            for (int m = 1; m < P; ++m) a = std::fma(T[m][k], f[(size_t)n * P + m], a);
            s_hat[n * P + k] = std::fma(t.L[k], tB[n], a);
            j_hat[n * P + k] = std::fma(t.L[k], dl, t.R[k] * dr);
        }
    }
}

static int apply_canonical(const fxo_grid* g, const Canon& c, const double* chi, const double* x, int normed, double* y) {
    const int P = g->P, Nx = g->Nx, Ny = g->Ny, nx = Nx * P, ny = Ny * P;
    size_t n = (size_t)nx * ny;
    std::vector<double> sx(n), jx(n), sy(n), jy(n);
    std::vector<double> u(std::max(nx, ny)), cw(std::max(nx, ny)), s(std::max(nx, ny)), jj(std::max(nx, ny));
    for (int r = 0; r < ny; ++r) {                 // x-lines
        int l = r % P;
        for (int cidx = 0; cidx < nx; ++cidx) { u[cidx] = x[(size_t)r * nx + cidx]; cw[cidx] = c.t.WW[l][cidx % P] * chi[(size_t)r * nx + cidx]; }
        line_ops(c.t, Nx, g->bcx, u.data(), cw.data(), s.data(), jj.data());
        for (int cidx = 0; cidx < nx; ++cidx) { sx[(size_t)r * nx + cidx] = s[cidx]; jx[(size_t)r * nx + cidx] = jj[cidx]; }
    }
    for (int cidx = 0; cidx < nx; ++cidx) {        // y-lines
        int k = cidx % P;
        for (int r = 0; r < ny; ++r) { u[r] = x[(size_t)r * nx + cidx]; cw[r] = c.t.WW[r % P][k] * chi[(size_t)r * nx + cidx]; }
        line_ops(c.t, Ny, g->bcy, u.data(), cw.data(), s.data(), jj.data());
        for (int r = 0; r < ny; ++r) { sy[(size_t)r * nx + cidx] = s[r]; jy[(size_t)r * nx + cidx] = jj[r]; }
    }
    for (int r = 0; r < ny; ++r) for (int cidx = 0; cidx < nx; ++cidx) {   // combine
        int l = r % P, k = cidx % P; size_t id = (size_t)r * nx + cidx;
        double t = c.JY[k] * jy[id];
        t = std::fma(c.JX[l], jx[id], t);
        t = std::fma(c.cyy, sy[id], t);
        t = std::fma(c.cxx, sx[id], t);
        if (normed) { double w = c.vol4 * c.t.WW[l][k]; double v = 1.0 / w; t = v * t; }
        y[id] = t;
    }
    return 0;
}

extern "C" int fxo_dg_apply_canonical(const fxo_grid* g, const double* chi, const double* x, int32_t normed, double* y) {
    if (!grid_ok(g) || x == y) return -1;
    Canon c; make_canon(g, c);
    return apply_canonical(g, c, chi, x, normed, y);
}

// ------------------------------------------------------------------------------------------------
// 6b. Stand-alone dG derivatives  y <- alpha * M x + beta * y,  M = d/dx or d/dy with forward, backward or
//     centred flux -- the paper's "dxdy" primitive ("derivatives in x and y", P:321 / Table 3, m = 3).
//     The paper gives no formulas (refs [21],[12]); reading (Q21): forward = F(N,h,bc) of section 5,
//     backward = -W^-1 F^T W (its negative W-adjoint), centred = (forward + backward)/2.
//     Definition: explicit matrices in 113-bit arithmetic.  Canonical fp64 order per line (cell n, node k):
//        a = chain_m(TT[k][m], u_{n,m});  a = fma(cP[k], tR_{n-1}, a);  a = fma(cN[k], tL_{n+1}, a);  d = RN((2/h) * a)
//        y = beta == 0 ? RN(alpha*d) : fma(alpha, d, RN(beta*y))
//     with TT = T (forward), -W^-1 T^T W (backward), their mean (centred); T = T0L in the first cell of a DIR line.
//     flux == 3: the stand-alone JUMP matrix (the paper's primitive is "y <- alpha M x + beta y" for the derivatives in x
//     and y "and jump" terms): M = Jhat(N, bc) of section 5, un-normed (sum over faces of [v][u]): block row
//     n has diagonal R R^T + L L^T, off-diagonals -R L^T (to n+1) and -L R^T (to n-1); no 2/h scale.  Canonical order: the
//     same three-step line with TT = R R^T + L L^T, cN = -R, cP = -L, s = 1.  Definition: build_J in 113-bit arithmetic.
// ------------------------------------------------------------------------------------------------

struct DTab { double TT[2][PMAX][PMAX], cN[PMAX], cP[PMAX]; };   // [0] interior, [1] first cell of a DIR line

static void make_dtab(int P, int flux, DTab& d) {
    RefElem e; ref_elem(P, e);
    if (flux == 3) {                                         // jump matrix (see above)
        for (int v = 0; v < 2; ++v) for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m)
            d.TT[v][k][m] = snap(e.R[k] * e.R[m] + e.L[k] * e.L[m]);
        for (int k = 0; k < P; ++k) { d.cN[k] = snap(-e.R[k]); d.cP[k] = snap(-e.L[k]); }
        return;
    }
    for (int v = 0; v < 2; ++v) for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) {
        auto T = [&](int a, int b) { q128 t = e.D[a][b] - e.R[a] * e.R[b] / e.w[a]; if (v) t += e.L[a] * e.L[b] / e.w[a]; return t; };
        q128 f = T(k, m), b = -T(m, k) * e.w[m] / e.w[k];
        q128 val = flux == 0 ? f : flux == 1 ? b : (f + b) / 2;
        d.TT[v][k][m] = snap(val);
    }
    for (int k = 0; k < P; ++k) {
        q128 cn = e.R[k] / e.w[k], cp = -e.L[k] / e.w[k];
        d.cN[k] = flux == 0 ? snap(cn) : flux == 1 ? 0.0 : snap(cn / 2);
        d.cP[k] = flux == 0 ? 0.0 : flux == 1 ? snap(cp) : snap(cp / 2);
    }
}

extern "C" int fxo_dg_dtables(int32_t P, int32_t flux, double* out) {      // TT[0], TT[1] (P*P each), cN, cP
    if (P < 1 || P > PMAX || flux < 0 || flux > 3) return -1;
    DTab d; make_dtab(P, flux, d);
    double* o = out;
    for (int v = 0; v < 2; ++v) for (int k = 0; k < P; ++k) for (int m = 0; m < P; ++m) *o++ = d.TT[v][k][m];
    for (int k = 0; k < P; ++k) *o++ = d.cN[k];
    for (int k = 0; k < P; ++k) *o++ = d.cP[k];
    return 0;
}

static void dline_canonical(const DTab& d, int P, int N, int bc, double s, const double* u, double* out) {
    std::vector<double> tL(N + 2), tR(N + 2);
    Tables t; make_tables(P, t);
    for (int n = 0; n < N; ++n) {
        double aL = t.L[0] * u[n * P], aR = t.R[0] * u[n * P];
        for (int m = 1; m < P; ++m) { aL = std::fma(t.L[m], u[n * P + m], aL); aR = std::fma(t.R[m], u[n * P + m], aR); }
        tL[n + 1] = aL; tR[n + 1] = aR;
    }
    if (bc == BC_PER) { tL[N + 1] = tL[1]; tR[0] = tR[N]; } else { tL[N + 1] = 0; tR[0] = 0; }
    for (int n = 0; n < N; ++n) {
        const double (*TT)[PMAX] = d.TT[(n == 0 && bc == BC_DIR) ? 1 : 0];
        for (int k = 0; k < P; ++k) {
            double a = TT[k][0] * u[n * P];
            for (int m = 1; m < P; ++m) a = std::fma(TT[k][m], u[n * P + m], a);
            a = std::fma(d.cP[k], tR[n], a);
            a = std::fma(d.cN[k], tL[n + 2], a);
            out[n * P + k] = s * a;
        }
    }
}

extern "C" int fxo_dg_derivative_canonical(const fxo_grid* g, int32_t dir, int32_t flux, double alpha, const double* x, double beta,
                                           double* y) {
    if (!grid_ok(g) || !deriv_bc_ok(g) || dir < 0 || dir > 1 || flux < 0 || flux > 3 || x == y) return -1;
    const int P = g->P, nx = g->Nx * P, ny = g->Ny * P;
    DTab d; make_dtab(P, flux, d);
    const int N = dir == 0 ? g->Nx : g->Ny, len = N * P, bc = dir == 0 ? g->bcx : g->bcy;
    const double h = dir == 0 ? g->lx / g->Nx : g->ly / g->Ny, s = flux == 3 ? 1.0 : 2.0 / h;
    std::vector<double> u(len), o(len);
    const int nl = dir == 0 ? ny : nx;
    for (int line = 0; line < nl; ++line) {
        for (int a = 0; a < len; ++a) u[a] = dir == 0 ? x[(size_t)line * nx + a] : x[(size_t)a * nx + line];
        dline_canonical(d, P, N, bc, s, u.data(), o.data());
        for (int a = 0; a < len; ++a) {
            size_t id = dir == 0 ? (size_t)line * nx + a : (size_t)a * nx + line;
            if (beta == 0.0) y[id] = alpha * o[a];
            else { double t = beta * y[id]; y[id] = std::fma(alpha, o[a], t); }
        }
    }
    return 0;
}

// definition: explicit matrices, 113 bit; M (rounded to double) is also returned for the numpy-side pins
extern "C" int fxo_dg_derivative_matrix_1d(int32_t N, int32_t P, double h, int32_t bc, int32_t flux, double* M_out) {
    if (bc != BC_PER && bc != BC_DIR) return -1;
    if (N < 1 || P < 1 || P > PMAX || !(h > 0) || flux < 0 || flux > 3) return -1;
    RefElem e; ref_elem(P, e);
    int n = N * P;
    if (flux == 3) {
        std::vector<q128> J; build_J(e, N, bc, J);
        for (size_t a = 0; a < (size_t)n * n; ++a) M_out[a] = (double)J[a];
        return 0;
    }
    std::vector<q128> F; build_F(e, N, (q128)h, bc, F);
    for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) {
        q128 f = F[(size_t)a * n + b], bk = -F[(size_t)b * n + a] * e.w[b % P] / e.w[a % P];
        M_out[(size_t)a * n + b] = (double)(flux == 0 ? f : flux == 1 ? bk : (f + bk) / 2);
    }
    return 0;
}

extern "C" int fxo_dg_derivative_definition(const fxo_grid* g, int32_t dir, int32_t flux, double alpha, const double* x, double beta,
                                            const double* y_in, double* y_out, double* scale) {
    if (!grid_ok(g) || !deriv_bc_ok(g) || dir < 0 || dir > 1 || flux < 0 || flux > 3) return -1;
    const int P = g->P, nx = g->Nx * P, ny = g->Ny * P;
    RefElem e; ref_elem(P, e);
    const int N = dir == 0 ? g->Nx : g->Ny, len = N * P, bc = dir == 0 ? g->bcx : g->bcy;
    q128 h = dir == 0 ? (q128)g->lx / g->Nx : (q128)g->ly / g->Ny;
    std::vector<q128> F, J;
    build_F(e, N, h, bc, F);
    if (flux == 3) build_J(e, N, bc, J);
    auto M = [&](int a, int b) {
        if (flux == 3) return J[(size_t)a * len + b];
        q128 f = F[(size_t)a * len + b], bk = -F[(size_t)b * len + a] * e.w[b % P] / e.w[a % P];
        return flux == 0 ? f : flux == 1 ? bk : (f + bk) / 2;
    };
    auto qabs = [](q128 v) { return v < 0 ? -v : v; };
    const int nl = dir == 0 ? ny : nx;
    for (int line = 0; line < nl; ++line) for (int a = 0; a < len; ++a) {
        q128 sum = 0, sa = 0;
        for (int b = 0; b < len; ++b) {
            q128 m = M(a, b);
            if (m != 0) { double xv = dir == 0 ? x[(size_t)line * nx + b] : x[(size_t)b * nx + line]; sum += m * xv; sa += qabs(m) * qabs((q128)xv); }
        }
        size_t id = dir == 0 ? (size_t)line * nx + a : (size_t)a * nx + line;
        q128 yv = beta == 0.0 ? (q128)0 : (q128)beta * y_in[id];
        y_out[id] = (double)((q128)alpha * sum + yv);
        if (scale) scale[id] = (double)(qabs((q128)alpha) * sa + qabs(yv));
    }
    return 0;
}

// ------------------------------------------------------------------------------------------------
// 6c. Fused pointwise product z <- alpha x1 y1 + beta x2 y2 + gamma z (added "to raise the work per call") and the
//     Arakawa bracket ("the Arakawa scheme [21]", the second composite the paper benchmarks, Fig. 6a: N = 9 calls).
//     Canonical order (Q22):  a = RN(alpha*x1); b = RN(beta*x2);
//         t = gamma == 0 ? RN(b*y2) : fma(b, y2, RN(gamma*z));   z = fma(a, y1, t).
//     Bracket {f,g} = df/dx dg/dy - df/dy dg/dx in Arakawa's conserving form, the mean of the three equivalent
//     expressions J1 = fx gy - fy gx, J2 = (f gy)_x - (f gx)_y, J3 = (g fx)_y - (g fy)_x, regrouped by outer derivative:
//         {f,g} = 1/3 [ fx gy - fy gx  +  Dx( f gy - g fy )  +  Dy( g fx - f gx ) ]      with centred dG derivatives,
//     evaluated as nine calls: 4 derivatives, 3 fused pointwise products, 2 accumulating derivatives.
// ------------------------------------------------------------------------------------------------
extern "C" void fxo_pointwise_dot2(double alpha, const double* x1, const double* y1, double beta, const double* x2, const double* y2,
                                   double gamma, double* z, int64_t n) {
    for (int64_t i = 0; i < n; ++i) {
        double a = alpha * x1[i], b = beta * x2[i], t;
        if (gamma == 0.0) t = b * y2[i];
        else { double gz = gamma * z[i]; t = std::fma(b, y2[i], gz); }
        z[i] = std::fma(a, y1[i], t);
    }
}

extern "C" int fxo_arakawa(const fxo_grid* g, const double* f, const double* gg, double* out) {
    if (!grid_ok(g) || !deriv_bc_ok(g)) return -1;
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P;
    std::vector<double> fx(n), fy(n), gx(n), gy(n), h1(n), h2(n);
    const double third = 1.0 / 3.0;
    fxo_dg_derivative_canonical(g, 0, 2, 1.0, f, 0.0, fx.data());
    fxo_dg_derivative_canonical(g, 1, 2, 1.0, f, 0.0, fy.data());
    fxo_dg_derivative_canonical(g, 0, 2, 1.0, gg, 0.0, gx.data());
    fxo_dg_derivative_canonical(g, 1, 2, 1.0, gg, 0.0, gy.data());
    fxo_pointwise_dot2(third, fx.data(), gy.data(), -third, fy.data(), gx.data(), 0.0, out, n);      // 1/3 (fx gy - fy gx)
    fxo_pointwise_dot2(third, f, gy.data(), -third, gg, fy.data(), 0.0, h1.data(), n);                // 1/3 (f gy - g fy)
    fxo_pointwise_dot2(third, gg, fx.data(), -third, f, gx.data(), 0.0, h2.data(), n);                // 1/3 (g fx - f gx)
    fxo_dg_derivative_canonical(g, 0, 2, 1.0, h1.data(), 1.0, out);                                  // += Dx(...)
    fxo_dg_derivative_canonical(g, 1, 2, 1.0, h2.data(), 1.0, out);                                  // += Dy(...)
    return 0;
}

// ------------------------------------------------------------------------------------------------
// 7. Preconditioned CG, step by step (Level-2 algorithm built from Level-1 calls only; the
//    exact dot "is for example important in a conjugate gradient method").  DESIGN.md 3.5.
//    Solves  div(chi grad phi) = rho  as  S phi = W o (-rho),  preconditioner V = 1/W.
// ------------------------------------------------------------------------------------------------

struct fxo_cg_info { int32_t iterations; int32_t status; double rel_residual; };
enum { FXO_OK = 0, FXO_MAXIT = 1, FXO_EINVAL = -1, FXO_EBREAKDOWN = -4 };

extern "C" int fxo_cg_solve(const fxo_grid* g, const double* chi, const double* rho, double* phi,
                            double tol, int32_t maxit, fxo_cg_info* info) {
    if (!grid_ok(g) || maxit < 0 || !(tol >= 0)) return FXO_EINVAL;
    Canon c; make_canon(g, c);
    const int64_t n = (int64_t)g->Nx * g->Ny * g->P * g->P;
    std::vector<double> W(n), V(n), rhs(n), r(n), z(n), p(n), q(n);
    fxo_dg_weights(g, W.data(), V.data());
    fxo_pointwise_dot(-1.0, W.data(), rho, 0.0, rhs.data(), n);
    apply_canonical(g, c, chi, phi, 0, q.data());
    r = rhs;
    fxo_axpby(-1.0, q.data(), 1.0, r.data(), n);
    fxo_pointwise_dot(1.0, V.data(), rhs.data(), 0.0, z.data(), n);
    double bz = fxo_exdot(rhs.data(), z.data(), n);
    int it = 0, status = FXO_OK;
    double rz = 0;
    if (bz == 0.0) {
        for (int64_t i = 0; i < n; ++i) phi[i] = 0.0;
        if (info) { info->iterations = 0; info->status = FXO_OK; info->rel_residual = 0.0; }
        return FXO_OK;
    }
    fxo_pointwise_dot(1.0, V.data(), r.data(), 0.0, z.data(), n);
    rz = fxo_exdot(r.data(), z.data(), n);
    p = z;
    double thresh = tol * std::sqrt(bz);
    if (!(std::sqrt(rz) <= thresh)) {
        status = FXO_MAXIT;
        for (it = 1; it <= maxit; ++it) {
            apply_canonical(g, c, chi, p.data(), 0, q.data());
            double pq = fxo_exdot(p.data(), q.data(), n);
            if (!(pq > 0.0) || !std::isfinite(pq)) { status = FXO_EBREAKDOWN; break; }
            double alpha = rz / pq;
            fxo_axpby(alpha, p.data(), 1.0, phi, n);
            fxo_axpby(-alpha, q.data(), 1.0, r.data(), n);
            fxo_pointwise_dot(1.0, V.data(), r.data(), 0.0, z.data(), n);
            double rz_new = fxo_exdot(r.data(), z.data(), n);
            if (std::sqrt(rz_new) <= thresh) { rz = rz_new; status = FXO_OK; break; }
            double beta = rz_new / rz;
            fxo_axpby(1.0, z.data(), beta, p.data(), n);
            rz = rz_new;
        }
        if (it > maxit) it = maxit;
    }
    if (info) { info->iterations = it; info->status = status; info->rel_residual = std::sqrt(rz) / std::sqrt(bz); }
    return status;
}

// ------------------------------------------------------------------------------------------------
// 8. 3-D product grids.  The paper's applications are "2D/3D drift-/gyro-fluid simulations"
//     with derivatives "on product spaces"; its elliptic equation is the PERPENDICULAR one,
//    div(chi grad_perp phi) = rho (Eq. 1c).  Reading DESIGN.md Q24: a 3-D product grid is
//    Nz planes of the 2-D grid with one node per plane in z (cell height hz = lz/Nz); a vector stores
//    plane after plane (idx3 = p*n2 + idx2); the operator acts in every plane and the planes meet only
//    in the dot products.  Weights (the volume form of the product space): W3 = RN(hz*W2), V3 = RN(1/W3).
//    Symmetric form S3 x = RN(hz * (S2 x_plane)); normed form A3 x = A2 x_plane (V3 o S3 = V2 o S2).
// ------------------------------------------------------------------------------------------------
struct fxo_grid3 { int32_t Nx, Ny, Nz, P; double lx, ly, lz; int32_t bcx, bcy; };
static bool grid3_ok(const fxo_grid3* g, fxo_grid* p) {
    if (!g || g->Nz < 1 || !(g->lz > 0)) return false;
    p->Nx = g->Nx; p->Ny = g->Ny; p->P = g->P; p->lx = g->lx; p->ly = g->ly; p->bcx = g->bcx; p->bcy = g->bcy;
    return grid_ok(p) != 0;
}

extern "C" int fxo_dg3_weights(const fxo_grid3* g, double* W, double* V) {
    fxo_grid p;
    if (!grid3_ok(g, &p)) return -1;
    const int64_t n2 = (int64_t)p.Nx * p.Ny * p.P * p.P;
    std::vector<double> W2(n2);
    fxo_dg_weights(&p, W2.data(), nullptr);
    const double hz = g->lz / g->Nz;
    for (int z = 0; z < g->Nz; ++z) for (int64_t i = 0; i < n2; ++i) {
        volatile double w = hz * W2[i];
        if (W) W[z * n2 + i] = w;
        if (V) V[z * n2 + i] = 1.0 / w;
    }
    return 0;
}

extern "C" int fxo_dg3_apply_canonical(const fxo_grid3* g, const double* chi, const double* x, int32_t normed, double* y) {
    fxo_grid p;
    if (!grid3_ok(g, &p)) return -1;
    const int64_t n2 = (int64_t)p.Nx * p.Ny * p.P * p.P;
    const double hz = g->lz / g->Nz;
    for (int z = 0; z < g->Nz; ++z) {
        fxo_dg_apply_canonical(&p, chi + z * n2, x + z * n2, normed, y + z * n2);
        if (!normed) for (int64_t i = 0; i < n2; ++i) { volatile double v = hz * y[z * n2 + i]; y[z * n2 + i] = v; }
    }
    return 0;
}

extern "C" int fxo_dg3_apply_definition(const fxo_grid3* g, const double* chi, const double* x, int32_t normed, double* y, double* scale) {
    fxo_grid p;
    if (!grid3_ok(g, &p)) return -1;
    const int64_t n2 = (int64_t)p.Nx * p.Ny * p.P * p.P;
    const q128 hz = (q128)g->lz / g->Nz;
    for (int z = 0; z < g->Nz; ++z)
        apply_definition_q(&p, chi + z * n2, x + z * n2, normed, normed ? (q128)1 : hz, y ? y + z * n2 : nullptr, scale ? scale + z * n2 : nullptr);
    return 0;
}

// PCG of section 7 with the 3-D primitives: one system over all planes (the dots are global).
extern "C" int fxo_cg3_solve(const fxo_grid3* g, const double* chi, const double* rho, double* phi,
                             double tol, int32_t maxit, fxo_cg_info* info) {
    fxo_grid pg;
    if (!grid3_ok(g, &pg) || maxit < 0 || !(tol >= 0)) return FXO_EINVAL;
    const int64_t n = (int64_t)pg.Nx * pg.Ny * pg.P * pg.P * g->Nz;
    std::vector<double> W(n), V(n), rhs(n), r(n), z(n), p(n), q(n);
    fxo_dg3_weights(g, W.data(), V.data());
    fxo_pointwise_dot(-1.0, W.data(), rho, 0.0, rhs.data(), n);
    fxo_dg3_apply_canonical(g, chi, phi, 0, q.data());
    r = rhs;
    fxo_axpby(-1.0, q.data(), 1.0, r.data(), n);
    fxo_pointwise_dot(1.0, V.data(), rhs.data(), 0.0, z.data(), n);
    double bz = fxo_exdot(rhs.data(), z.data(), n);
    int it = 0, status = FXO_OK;
    double rz = 0;
    if (bz == 0.0) {
        for (int64_t i = 0; i < n; ++i) phi[i] = 0.0;
        if (info) { info->iterations = 0; info->status = FXO_OK; info->rel_residual = 0.0; }
        return FXO_OK;
    }
    fxo_pointwise_dot(1.0, V.data(), r.data(), 0.0, z.data(), n);
    rz = fxo_exdot(r.data(), z.data(), n);
    p = z;
    double thresh = tol * std::sqrt(bz);
    if (!(std::sqrt(rz) <= thresh)) {
        status = FXO_MAXIT;
        for (it = 1; it <= maxit; ++it) {
            fxo_dg3_apply_canonical(g, chi, p.data(), 0, q.data());
            double pq = fxo_exdot(p.data(), q.data(), n);
            if (!(pq > 0.0) || !std::isfinite(pq)) { status = FXO_EBREAKDOWN; break; }
            double alpha = rz / pq;
            fxo_axpby(alpha, p.data(), 1.0, phi, n);
            fxo_axpby(-alpha, q.data(), 1.0, r.data(), n);
            fxo_pointwise_dot(1.0, V.data(), r.data(), 0.0, z.data(), n);
            double rz_new = fxo_exdot(r.data(), z.data(), n);
            if (std::sqrt(rz_new) <= thresh) { rz = rz_new; status = FXO_OK; break; }
            double beta = rz_new / rz;
            fxo_axpby(1.0, z.data(), beta, p.data(), n);
            rz = rz_new;
        }
        if (it > maxit) it = maxit;
    }
    if (info) { info->iterations = it; info->status = status; info->rel_residual = std::sqrt(rz) / std::sqrt(bz); }
    return status;
}
