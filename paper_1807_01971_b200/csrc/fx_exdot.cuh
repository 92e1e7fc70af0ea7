// fx_exdot.cuh -- device side of the exactly rounded dot product (section 3.1).
//
// The paper's scheme: TwoProd splits every product error-free into (p, e); p and e are accumulated in
// floating-point expansions held in registers; what an expansion cannot hold goes to a long accumulator
// ("a very long fixed point number") which is "rarely invoked"; partial results are merged
// "on various levels" and rounded once.
//
// What is kept and what differs on sm_100a:
//   * kept: TwoProd by FMA, register-resident expansions in front of an integer long accumulator, integer
//     merging (associative -> result independent of thread, warp, block and grid shape);
//   * differs: the expansion is a BINNED one.  A warp keeps a common window top 2^T; bin k is a double S[k] that
//     sits in the binade [2^(E_k+52), 2^(E_k+53)], E_k = T - W*(k+1), so that ulp(S[k]) = 2^E_k.  Adding a value
//     v (|v| <= |S[k]|) is FastTwoSum(S[k], v):  s = S[k]+v; q = s-S[k]; r = v-q  -- always error-free; r
//     (|r| <= 2^(E_k-1)) drops into the next bin.  That is 3 fp64 operations per bin and value instead of the
//     6 of a TwoSum, with no data-dependent branch in the common case, which is what fits B200's ratio of
//     ~2.3 fp64 issue slots per HBM byte.  A non-zero remainder below the last bin, and products outside the
//     range where TwoProd is error-free, take a slow path that deposits exact integer chunks into the shared
//     long accumulator.
//
// Long accumulator: 136 signed 64-bit digits spaced 32 bit apart, digit d weighs 2^(32 d - 2176) (the same
// fixed-point grid as 68 limbs x 64 bit with the LSB at 2^-2176: below the smallest product bit 2^-2148, above
// 2^2048 * n).  One copy in shared memory per CTA, one in global memory per context.

#ifndef FX_EXDOT_CUH
#define FX_EXDOT_CUH

#include <stdint.h>

#define FX_NDIG 136
#define FX_NLIMB 68
#define FX_BIAS 2176
#define FX_FLAG_NAN 1
#define FX_FLAG_PINF 2
#define FX_FLAG_NINF 4

typedef unsigned long long fx_u64;

struct ExShared {
    fx_u64 dig[FX_NDIG];     // signed digits, two's complement wrap-around arithmetic
    fx_u64 lim[FX_NLIMB];    // last CTA only: the canonical limbs while they are normalised and rounded
    int flags;
    int is_last;
    int dlo, dhi;            // last CTA only: range of non-zero merged digits
    double res;              // ex_grid_reduce: the rounded value, broadcast to the CTA
    unsigned int stat[4];    // slow-path census of this CTA: exact-double deposits, integer-product deposits, window moves
    int gflags;              // last CTA only: the merged flags, fetched together with the digits
};

struct ExGlobal {            // device scratch of one context
    fx_u64* dig;             // [FX_NDIG]   merged CTA digits of the running launch (zero between launches)
    fx_u64* limbs;           // [FX_NLIMB]  canonical two's complement accumulator of the running call
    int* flags;              // [1]
    unsigned int* ticket;    // [1]         CTAs finished (zero between launches)
    fx_u64* stats;           // [4]         slow-path census since the last reset (fx_exdot_stats): how rarely the long
                             //             accumulator is "invoked"
    int keep_limbs;          // write the canonical limbs back after the last launch of a call (fx_exdot_digits); a plain dot
                             // only needs its rounded value and skips that store and its fence
};

// 64-bit add into a shared-memory word.  Shared memory has no native 64-bit atomic add (atomicAdd compiles to a compare-and-swap
// spin, ATOMS.CAST.SPIN.64, which collapses when many lanes hit the few digits of one exponent region); two native 32-bit adds
// do the same: the low add returns the old value, from which THIS adder knows whether it caused the wrap-around, and carries
// it into the high word.  Every wrap is seen by exactly one adder, so the 64-bit total is exact in any order.
__device__ __forceinline__ void ex_sadd64(fx_u64* p, fx_u64 v) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(p);
    const unsigned lo = (unsigned)v;
    unsigned hi = (unsigned)(v >> 32);
    if (lo) {
        unsigned old;
        asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old) : "r"(a), "r"(lo) : "memory");
        hi += (old + lo) < old ? 1u : 0u;
    }
    if (hi) asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(a + 4u), "r"(hi) : "memory");
}

// add (-1)^neg * (hi:lo) * 2^(b - FX_BIAS) into the CTA's digit array in shared memory.
// The (up to) five 64-bit adds of ex_sadd64 with their atomics in two rounds -- all the low-word adds (each returns the
// old value), then all the high-word adds with the wrap-around carries: one shared-memory round trip instead of five in a
// row (the volatile asm statements keep their order, so written one digit after the other every low add waited for
// the one before: 0.3 us per deposit, 2 us per flush of a warp's six bins).
__device__ __forceinline__ void ex_deposit(fx_u64* dig, int b, fx_u64 hi, fx_u64 lo, bool neg) {
    const int d = b >> 5, s = b & 31;
    fx_u64 w0 = lo << s;
    fx_u64 w1 = (hi << s) | (s ? (lo >> (64 - s)) : 0ull);
    fx_u64 w2 = s ? (hi >> (64 - s)) : 0ull;
    fx_u64 c[5] = {w0 & 0xffffffffull, w0 >> 32, w1 & 0xffffffffull, w1 >> 32, w2};
    const unsigned a0 = (unsigned)__cvta_generic_to_shared(&dig[d]);
    unsigned vlo[5], vhi[5], old[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const fx_u64 v = neg ? (0ull - c[i]) : c[i];
        vlo[i] = (unsigned)v; vhi[i] = (unsigned)(v >> 32); old[i] = 0u;
        if (vlo[i]) asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(old[i]) : "r"(a0 + 8u * i), "r"(vlo[i]) : "memory");
    }
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const unsigned h = vhi[i] + ((old[i] + vlo[i]) < old[i] ? 1u : 0u);
        if (h) asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(a0 + 8u * i + 4u), "r"(h) : "memory");
    }
}

// any finite double v (exactly), DESIGN.md 6.1 "slow path 1"
static __device__ __noinline__ void ex_deposit_double(ExShared* sh, double v) {
    const fx_u64 bits = (fx_u64)__double_as_longlong(v);
    const int be = (int)((bits >> 52) & 0x7ff);
    fx_u64 m = bits & 0xfffffffffffffull;
    if (be) m |= 1ull << 52;
    if (m == 0) return;
    const int E = (be ? be : 1) - 1075;
    atomicAdd(&sh->stat[0], 1u);
    ex_deposit(sh->dig, E + FX_BIAS, 0ull, m, (bits >> 63) != 0);
}

// exact product of any two doubles, DESIGN.md 6.1 "slow path 2": integer mantissa product (106 bit)
static __device__ __noinline__ void ex_deposit_product(ExShared* sh, double x, double y) {
    const fx_u64 bx = (fx_u64)__double_as_longlong(x), by = (fx_u64)__double_as_longlong(y);
    const int ex = (int)((bx >> 52) & 0x7ff), ey = (int)((by >> 52) & 0x7ff);
    const fx_u64 fx = bx & 0xfffffffffffffull, fy = by & 0xfffffffffffffull;
    const bool neg = ((bx ^ by) >> 63) != 0;
    if (ex == 0x7ff || ey == 0x7ff) {
        const bool nan = (ex == 0x7ff && fx) || (ey == 0x7ff && fy) || (ex == 0 && fx == 0) || (ey == 0 && fy == 0);
        atomicOr(&sh->flags, nan ? FX_FLAG_NAN : (neg ? FX_FLAG_NINF : FX_FLAG_PINF));
        return;
    }
    const fx_u64 mx = ex ? (fx | (1ull << 52)) : fx, my = ey ? (fy | (1ull << 52)) : fy;
    const fx_u64 lo = mx * my, hi = __umul64hi(mx, my);
    if ((lo | hi) == 0) return;
    atomicAdd(&sh->stat[1], 1u);
    const int E = (ex ? ex : 1) + (ey ? ey : 1) - 2150;          // value = mx*my * 2^E, E >= -2148
    ex_deposit(sh->dig, E + FX_BIAS, hi, lo, neg);
}

__device__ __forceinline__ long long ex_warp_sum(long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// lane 0 of a warp: add c * 2^(E - FX_BIAS + FX_BIAS) ... i.e. the signed count c at bit position b
static __device__ __noinline__ void ex_deposit_count(ExShared* sh, int b, long long c) {
    ex_deposit(sh->dig, b, 0ull, (fx_u64)(c < 0 ? -c : c), c < 0);
}

// Per-thread binned expansion with a warp-uniform window.  K bins of W bit.  All members are inlined so that the
// state lives in registers; only the integer deposits are calls.
// KL further bins below the K of the hot chain (a "low window"): they are visited only by a thread whose batch left a
// remainder below the first K*W bits -- data whose exponents spread over more than the window (config 1's condition
// targets 1e32 and 1e40: products over 2^-53 .. 2^53 plus their 106 bits).  Without them every such remainder went to the
// shared long accumulator with atomics: 0.5 deposits per element at 1e40 and 234 GB/s instead of 6800.
template <int K, int W, int KL = 0>
struct ExAcc {
    static constexpr int KT = K + KL;
    static constexpr int CAP = 1 << (50 - W);            // deposits per bin before S[k] must be re-centred
    static constexpr int MARGIN = 6;                     // head-room (bit) above the largest product seen
    static constexpr int TB_MIN = -1074 + KT * W + 1022; // lowest bin stays a normal double with ulp >= 2^-1074
    static constexpr unsigned BE_LO = 63;                // fast path: 2^-960 <= |p| < 2^1000 (TwoProd error-free,
    static constexpr unsigned BE_HI = 2022;              //   no overflow of the top bin)
    double S[KT];
    long long C[KT];
    int Tb;          // T + 1022; |p| < 2^T  <=>  biased exponent of p <= Tb.   very negative = no window yet
    int cnt, ren;

    __device__ __forceinline__ void init() {
#pragma unroll
        for (int k = 0; k < KT; ++k) { S[k] = 0.0; C[k] = 0; }
        Tb = -(1 << 29); cnt = 0; ren = 0;
    }
    __device__ __forceinline__ long long mbits(int k) const {      // bit pattern of 1.5 * 2^(E_k + 52)
        const int be = Tb - 1022 - W * (k + 1) + 52 + 1023;
        return ((long long)be << 52) | (1ll << 51);
    }
    __device__ __forceinline__ void recentre() {                    // S[k] -> centre, integer part -> C[k]
#pragma unroll
        for (int k = 0; k < KT; ++k) {
            const long long m = mbits(k);
            C[k] += __double_as_longlong(S[k]) - m;                 // same binade: bit patterns are linear in value
            S[k] = __longlong_as_double(m);
        }
        cnt = 0; ++ren;
    }
    // all 32 lanes: merge the warp's bins by shuffles (the KT butterflies interleaved), then lane k deposits bin k into the
    // CTA's long accumulator -- the KT deposits run side by side in one call instead of one after the other in lane 0
    __device__ __forceinline__ void flush(ExShared* sh) {
        if (Tb > -(1 << 28)) {
            long long c[KT];
#pragma unroll
            for (int k = 0; k < KT; ++k) c[k] = C[k] + (__double_as_longlong(S[k]) - mbits(k));
#pragma unroll
            for (int o = 16; o > 0; o >>= 1)
#pragma unroll
                for (int k = 0; k < KT; ++k) c[k] += __shfl_xor_sync(0xffffffffu, c[k], o);
            const int lane = threadIdx.x & 31;
            long long mine = 0;
#pragma unroll
            for (int k = 0; k < KT; ++k) mine = lane == k ? c[k] : mine;
            if (lane < KT && mine != 0) ex_deposit_count(sh, Tb - 1022 - W * (lane + 1) + FX_BIAS, mine);
#pragma unroll
            for (int k = 0; k < KT; ++k) { C[k] = 0; S[k] = __longlong_as_double(mbits(k)); }
        }
        cnt = 0; ren = 0;
    }
    __device__ __forceinline__ void reanchor(ExShared* sh, int bemax) {
        if ((threadIdx.x & 31) == 0 && Tb > -(1 << 28)) atomicAdd(&sh->stat[2], 1u);      // (the first anchoring of a warp is not a move)
        flush(sh);
        const int t = bemax + MARGIN;
        Tb = t < TB_MIN ? TB_MIN : t;
#pragma unroll
        for (int k = 0; k < KT; ++k) { S[k] = __longlong_as_double(mbits(k)); C[k] = 0; }
    }

    // U products per lane; must be called by all 32 lanes of the warp together.  Elements with active == false must
    // pass x = y = 0 (padding); they are not inspected.  ALLACT: every element is active (no selects).
    // Instruction budget per element: 2 + 3K + 3(K-1) fp64 operations and ~5 integer ones; the range
    // test and the below-window test are OR/MAX-reduced over the batch and branch once per batch.
    // NOERR: the caller guarantees that every product is exact in fp64 (y = 1: the exact sum), so e = 0 is not carried.
    template <int U, bool ALLACT, bool NOERR = false>
    __device__ __forceinline__ void add(const double (&x)[U], const double (&y)[U], const bool (&active)[U], ExShared* sh) {
        constexpr unsigned LOS = BE_LO << 20, RANGES = (BE_HI - BE_LO) << 20;
        double p[U], e[U];
        unsigned tmax = 0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            p[u] = __dmul_rn(x[u], y[u]);
            e[u] = NOERR ? 0.0 : __fma_rn(x[u], y[u], -p[u]);        // TwoProd
            unsigned hp = (unsigned)__double2hiint(p[u]) & 0x7ff00000u;
            if (!ALLACT) hp = active[u] ? hp : LOS;
            const unsigned t = hp - LOS;                             // wraps to huge below the range
            tmax = t > tmax ? t : tmax;
        }
        if (tmax > RANGES) {                                         // some product outside TwoProd's error-free range, or zero
            tmax = 0;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const unsigned be = ((unsigned)__double2hiint(p[u]) >> 20) & 0x7ffu;
                const bool act = ALLACT || active[u];
                if (act && (be - BE_LO) > (BE_HI - BE_LO)) {
                    const bool xz = (((unsigned)__double2hiint(x[u]) & 0x7fffffffu) | (unsigned)__double2loint(x[u])) == 0u;
                    const bool yz = (((unsigned)__double2hiint(y[u]) & 0x7fffffffu) | (unsigned)__double2loint(y[u])) == 0u;
                    if (be == 0x7ffu || !(xz || yz)) ex_deposit_product(sh, x[u], y[u]);
                    p[u] = 0.0; e[u] = 0.0;
                } else if (act) {
                    const unsigned t = (be - BE_LO) << 20;
                    tmax = t > tmax ? t : tmax;
                }
            }
        }
        const int bemax = (int)(tmax >> 20) + (int)BE_LO;
        if (__any_sync(0xffffffffu, bemax > Tb)) reanchor(sh, __reduce_max_sync(0xffffffffu, bemax));
        if (cnt + U > CAP) { recentre(); if (ren >= 32) flush(sh); }
        cnt += U;
        unsigned rlo = 0, rhi = 0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            double v = p[u], w = e[u];
#pragma unroll
            for (int k = 0; k < K; ++k) {
                const double s = __dadd_rn(S[k], v);
                const double q = __dsub_rn(s, S[k]);
                v = __dsub_rn(v, q);
                S[k] = s;
            }
#pragma unroll
            for (int k = NOERR ? K : 1; k < K; ++k) {                // |e| < ulp(S[0])/2: bin 0 cannot take any of it
                const double s = __dadd_rn(S[k], w);
                const double q = __dsub_rn(s, S[k]);
                w = __dsub_rn(w, q);
                S[k] = s;
            }
            p[u] = v; e[u] = w;
            rlo |= (unsigned)__double2loint(v) | (unsigned)__double2loint(w);
            rhi |= (unsigned)__double2hiint(v) | (unsigned)__double2hiint(w);
        }
        if (KL > 0 && (rlo | (rhi & 0x7fffffffu))) {                 // bits below the hot chain's K*W bits: the low window
            rlo = 0; rhi = 0;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                double v = p[u], w = e[u];
#pragma unroll
                for (int k = K; k < KT; ++k) {
                    const double s = __dadd_rn(S[k], v);
                    const double q = __dsub_rn(s, S[k]);
                    v = __dsub_rn(v, q);
                    const double s2 = NOERR ? s : __dadd_rn(s, w);
                    const double q2 = NOERR ? 0.0 : __dsub_rn(s2, s);
                    if (!NOERR) w = __dsub_rn(w, q2);
                    S[k] = s2;
                }
                p[u] = v; e[u] = w;
                rlo |= (unsigned)__double2loint(v) | (unsigned)__double2loint(w);
                rhi |= (unsigned)__double2hiint(v) | (unsigned)__double2hiint(w);
            }
        }
        if (rlo | (rhi & 0x7fffffffu)) {                             // bits below the window: exact, but slow
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (p[u] != 0.0) ex_deposit_double(sh, p[u]);
                if (e[u] != 0.0) ex_deposit_double(sh, e[u]);
            }
        }
    }
    template <int U>
    __device__ __forceinline__ void add(const double (&x)[U], const double (&y)[U], const bool (&active)[U], ExShared* sh) {
        add<U, false>(x, y, active, sh);
    }
    template <int U>
    __device__ __forceinline__ void add_all(const double (&x)[U], const double (&y)[U], ExShared* sh) {
        bool act[U];
#pragma unroll
        for (int u = 0; u < U; ++u) act[u] = true;
        add<U, true>(x, y, act, sh);
    }
};

__device__ __forceinline__ void ex_shared_init(ExShared* sh) {
    for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) sh->dig[i] = 0ull;
    if (threadIdx.x == 0) { sh->flags = 0; sh->is_last = 0; }
    if (threadIdx.x < 4) sh->stat[threadIdx.x] = 0u;
    __syncthreads();
}

// ---- final stage, one thread: merge digits into the canonical limbs, round once ----------------------------

// RN(limbs) with ties to even, gradual underflow, overflow to inf; exact zero -> +0.0   (DESIGN.md 3.1 step 4).
// Only limbs [a, bb] are inspected: limbs below a are zero, limbs above bb repeat the sign of limb bb.
__device__ inline double ex_round(const fx_u64* limbs, int flags, fx_u64* mag /* scratch [FX_NLIMB] */, int a, int bb) {
    if ((flags & FX_FLAG_NAN) || ((flags & FX_FLAG_PINF) && (flags & FX_FLAG_NINF)))
        return __longlong_as_double(0x7FF8000000000000ll);
    if (flags & FX_FLAG_PINF) return __longlong_as_double(0x7FF0000000000000ll);
    if (flags & FX_FLAG_NINF) return __longlong_as_double((long long)0xFFF0000000000000ull);
    const bool neg = (limbs[bb] >> 63) != 0;
    fx_u64 carry = neg ? 1ull : 0ull;
    int top = -1;
    for (int k = a; k <= bb; ++k) {
        const fx_u64 v = neg ? ~limbs[k] : limbs[k];
        const fx_u64 s = v + carry;
        carry = (s < v) ? 1ull : 0ull;
        mag[k] = s;
        if (s) top = k;
    }
    if (top < 0) return 0.0;
#define FX_MAG(k) (((k) >= a && (k) <= bb) ? mag[(k)] : 0ull)
    const int t = 64 * top + 63 - __clzll((long long)mag[top]);
    const int PMIN = -1074 + FX_BIAS;
    const bool normal = (t - 52) >= PMIN;
    const int p = normal ? (t - 52) : PMIN;
    fx_u64 mant;                                                      // bits [p, p+63] (all above t are zero): < 2^53
    {
        const int k = p >> 6, sft = p & 63;
        mant = FX_MAG(k) >> sft;
        if (sft) mant |= FX_MAG(k + 1) << (64 - sft);
    }
    const fx_u64 round_bit = (FX_MAG((p - 1) >> 6) >> ((p - 1) & 63)) & 1ull;
    bool sticky = false;
    {
        const int b = p - 1;                                          // bits [0, b) below the round bit
        const int k = b >> 6, sft = b & 63;
        for (int i = a; i < k && i <= bb; ++i) sticky |= (mag[i] != 0);
        if (sft) sticky |= (FX_MAG(k) & ((1ull << sft) - 1ull)) != 0;
    }
#undef FX_MAG
    if (round_bit && (sticky || (mant & 1ull))) mant += 1ull;
    fx_u64 bits;
    if (normal) {
        const long long be = (long long)(t - FX_BIAS) + 1023;
        if (be >= 2047) bits = 0x7FF0000000000000ull;
        else bits = ((fx_u64)be << 52) + (mant - (1ull << 52));       // mant == 2^53 carries into the exponent
    } else bits = mant;                                               // mant == 2^52 is the smallest normal
    if (neg) bits |= 1ull << 63;
    return __longlong_as_double((long long)bits);
}

// End of a CTA: digits -> global, the last CTA to arrive finalises (single pass, no second launch): its threads fetch
// the merged digits and the running limbs in parallel, thread 0 carry-normalises them in shared memory and rounds
// once.  Returns true in every thread of the last CTA after the result has been written.
// `first`/`last`: position of this launch in a multi-launch call (first: limbs start from zero; last: round).
__device__ __forceinline__ bool ex_block_finish(ExShared* sh, const ExGlobal& g, int first, int last, double* result) {
    __syncthreads();
    const bool solo = gridDim.x * gridDim.y == 1;                  // one CTA: its shared digits ARE the merged digits -- no
    if (!solo) {                                                     // global round trips at all (the latency of a small dot)
        for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) {
            const fx_u64 v = sh->dig[i];
            if (v) atomicAdd(&g.dig[i], v);
        }
    }
    if (threadIdx.x == 0 && sh->flags && !(solo && first && last)) atomicOr(g.flags, sh->flags);
    if (threadIdx.x < 4 && sh->stat[threadIdx.x]) atomicAdd(&g.stats[threadIdx.x], (fx_u64)sh->stat[threadIdx.x]);
    if (!solo) {
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned int t = atomicAdd(g.ticket, 1u);
            sh->is_last = (t == gridDim.x * gridDim.y - 1);
        }
        __syncthreads();
        if (!sh->is_last) return false;
        __threadfence();
    }
    if (threadIdx.x == 0) { sh->dlo = FX_NDIG; sh->dhi = -1; }
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) sh->gflags = (solo && first && last) ? sh->flags : __ldcg(g.flags);   // with the digits: one round trip
    for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) {
        const fx_u64 v = solo ? sh->dig[i] : __ldcg(&g.dig[i]);
        if (!solo) { sh->dig[i] = v; if (v) g.dig[i] = 0ull; }
        if (v) { atomicMin(&sh->dlo, i); atomicMax(&sh->dhi, i); }
    }
    for (int i = threadIdx.x; i < FX_NLIMB; i += blockDim.x) sh->lim[i] = first ? 0ull : __ldcg(&g.limbs[i]);
    __syncthreads();
    // thread 0: carry-normalise.  In the first launch of a call the limbs start from zero, so only the limbs that hold
    // non-zero digits (a handful: the data's exponent window) need the serial pass; above them the sign repeats.
    if (threadIdx.x == 0) {
        int la = 0, lb = FX_NLIMB - 1;
        if (first) { la = sh->dhi < 0 ? 0 : (sh->dlo >> 1); lb = sh->dhi < 0 ? 0 : (sh->dhi >> 1); }
        long long carry = 0;
        fx_u64 c2 = 0;
        int k = la;
        for (; k < FX_NLIMB; ++k) {
            if (k > lb && first && (carry == 0 || carry == -1) && c2 == 0) break;   // nothing but sign extension left
            long long v = (long long)sh->dig[2 * k] + carry;
            const fx_u64 lo = (fx_u64)v & 0xffffffffull;
            carry = v >> 32;
            v = (long long)sh->dig[2 * k + 1] + carry;
            const fx_u64 hi = (fx_u64)v & 0xffffffffull;
            carry = v >> 32;
            const fx_u64 word = lo | (hi << 32);
            const fx_u64 old = sh->lim[k];
            const fx_u64 s1 = old + word;
            fx_u64 c = (s1 < old) ? 1ull : 0ull;
            const fx_u64 s2 = s1 + c2;
            c |= (s2 < s1) ? 1ull : 0ull;
            c2 = c;
            sh->lim[k] = s2;
        }
        // k = first limb not written; limbs k.. are 0 (carry 0) or all ones (carry -1)
        const fx_u64 fill = (carry == -1) ? ~0ull : 0ull;
        int bb = k;
        if (k < FX_NLIMB) sh->lim[k] = fill; else bb = FX_NLIMB - 1;
        sh->dlo = k; sh->dhi = (carry == -1) ? 1 : 0;                 // hand the fill range to the other threads
        if (last) {
            const int flags = sh->gflags;
            g.flags[1] = flags;                       // kept for fx_exdot_digits
            if (!(solo && first)) g.flags[0] = 0;
            if (result) *result = ex_round(sh->lim, flags, sh->dig, la, bb);
        }
        if (!solo) *g.ticket = 0u;
    }
    if (last && !g.keep_limbs) return true;                           // (uniform: nobody needs the limbs of a finished plain dot)
    __syncthreads();
    {
        const int kf = sh->dlo;
        const fx_u64 fill = sh->dhi ? ~0ull : 0ull;
        for (int i = threadIdx.x; i < FX_NLIMB; i += blockDim.x) g.limbs[i] = (i > kf) ? fill : sh->lim[i];
    }
    __threadfence();
    __syncthreads();
    return true;
}

// Thread 0 of a CTA: sh->dig holds merged digits (range dlo..dhi), limbs start from zero -> RN(value).
__device__ inline double ex_round_digits_shared(ExShared* sh, int flags) {
    const int la = sh->dhi < 0 ? 0 : (sh->dlo >> 1), lb = sh->dhi < 0 ? 0 : (sh->dhi >> 1);
    long long carry = 0;
    int k = la;
    for (; k < FX_NLIMB; ++k) {
        if (k > lb && (carry == 0 || carry == -1)) break;
        long long v = (long long)sh->dig[2 * k] + carry;
        const fx_u64 lo = (fx_u64)v & 0xffffffffull;
        carry = v >> 32;
        v = (long long)sh->dig[2 * k + 1] + carry;
        const fx_u64 hi = (fx_u64)v & 0xffffffffull;
        carry = v >> 32;
        sh->lim[k] = lo | (hi << 32);
    }
    int bb = k;
    if (k < FX_NLIMB) sh->lim[k] = (carry == -1) ? ~0ull : 0ull; else bb = FX_NLIMB - 1;
    return ex_round(sh->lim, flags, sh->dig, la, bb);
}

// The two halves of a reduction that is finished by its CONSUMER (the fused CG kernels): a kernel's CTAs
// only add their digits to a global digit buffer (ex_publish: no ticket, no last-CTA finaliser, no tail), and every CTA
// of the NEXT kernel fetches the merged digits and normalises and rounds them itself (ex_fetch_round) while its first
// tiles are already in flight -- all CTAs hold the same bits.  gdig/gflags must be zero before the producing kernel.
__device__ __forceinline__ void ex_publish(ExShared* sh, fx_u64* gdig, int* gflags, fx_u64* gstats) {
    __syncthreads();
    for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) {
        const fx_u64 v = sh->dig[i];
        if (v) atomicAdd(&gdig[i], v);
    }
    if (threadIdx.x == 0 && sh->flags) atomicOr(gflags, sh->flags);
    if (threadIdx.x < 4 && sh->stat[threadIdx.x]) atomicAdd(&gstats[threadIdx.x], (fx_u64)sh->stat[threadIdx.x]);
}
__device__ inline double ex_round_digits_shared(ExShared* sh, int flags);
__device__ __forceinline__ double ex_fetch_round(ExShared* sh, const fx_u64* gdig, const int* gflags) {
    if (threadIdx.x == 0) { sh->dlo = FX_NDIG; sh->dhi = -1; }
    __syncthreads();
    if (threadIdx.x == blockDim.x - 1) sh->flags = __ldcg(gflags);  // (in the same round trip as the digits)
    for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) {
        const fx_u64 v = __ldcg(&gdig[i]);
        sh->dig[i] = v;
        if (v) { atomicMin(&sh->dlo, i); atomicMax(&sh->dhi, i); }
    }
    __syncthreads();
    if (threadIdx.x == 0) sh->res = ex_round_digits_shared(sh, sh->flags);
    __syncthreads();
    return sh->res;
}

// Grid-wide exact reduction inside a cooperative (persistent) kernel: every CTA adds its digits to gdig, the grid
// synchronises, and EVERY CTA normalises and rounds the merged digits itself, so that all of them hold the same bits
// without a second synchronisation.  gdig/gflags must be zero on entry; the caller re-zeroes them one phase later
// (DESIGN.md 6.5).  `gsync` is cooperative_groups::grid_group::sync.
template <class GRID>
__device__ __forceinline__ double ex_grid_reduce(ExShared* sh, fx_u64* gdig, int* gflags, GRID& grid) {
    __syncthreads();
    for (int i = threadIdx.x; i < FX_NDIG; i += blockDim.x) {
        const fx_u64 v = sh->dig[i];
        if (v) atomicAdd(&gdig[i], v);
    }
    if (threadIdx.x == 0 && sh->flags) atomicOr(gflags, sh->flags);
    grid.sync();                                  // (fences: the digits of every CTA are visible after it)
    return ex_fetch_round(sh, gdig, gflags);      // digits and flags in one round trip, one thread normalises and rounds
}

#endif
