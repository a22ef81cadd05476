// afs_long.cuh -- the LONG class: EK / CARD longer than 64 literals.  warp = (constraint, restart), CTA = one
// constraint x one tile of 32 restarts.  Count basis (G10):
//
//   Q(z) = prod_j (u_j + p_j z),  u = (1+y)/2, p = (1-y)/2,  q_t = [z^t] Q = Pr[t literals true]
//
//   classes   a literal on the boundary of the cube is the factor 1 (y = +1) or z (y = -1): an exact shift of the pmf,
//             no arithmetic.  PGD iterates sit on that boundary in most coordinates (clipping; fixed variables,
//             P:L140), so the pmf is built from the INTERIOR literals only:  Q(z) = z^nB0 * Qred(z),  deg Qred = Leff.
//             Which literals are interior, and which way they lean, is read from two bit words per (variable, tile of
//             32 restarts) that the variable pass writes with the iterate: sign (x < 0) and saturated (|x| = 1).
//   ratios    per interior literal R = min(u, p) / max(u, p) in (0, 1] (type A: p <= 1/2, type B: p > 1/2);
//             max(u, p) = 1 / (1 + R) because u + p = 1.
//   lists     the interior literals of a restart are compacted into  [ B interior | A interior ], both sections padded
//             with neutral R = 0 entries to multiples of four.
//   forward   Qred = rev(prod_B (1 + R_j w)) * prod_A (1 + R_j z) / prod (1 + R_j): every literal is the one-FMA
//             update q_t += R q_{t-1}; after the B section the coefficient vector is reversed once (prod_B (z + R_j)
//             is the reversal of prod_B (1 + R_j w)).  The scalar 1 / prod (1 + R_j) is applied every 32 literals
//             (growth inside a block <= 2^32).  The pmf lives in registers, cell t = (row*32 + lane)*4 + c; rows that
//             are still identically zero are skipped (warp-uniform).
//   gradient  dFE/dy_j = sum_t d_t q_t^(-j) with at most two non-zero d_t.  q^(-j) comes from q by removing
//             literal j in the STABLE direction: s_t = q_t - R_j s_{t-1} from the bottom for type A, the same
//             recurrence from the top for type B; q^(-j) = (1 + R_j) s.  Nothing that vanishes at x = +-1 is ever
//             divided by (BASELINE.json subsystem (2)).  A warp runs chains of one direction and one length; every
//             lane carries up to four chains that share each broadcast load of q.  Boundary literals need no chain:
//             q^(-j) = q (y = +1) or q shifted by one (y = -1) -- one pair of values per (constraint, restart).
// The reduced pmf sits in shared memory at A[off + t] with off = (3 - Leff) mod 4, so that the top-down chains read
// aligned 16-byte blocks from index 0 and the bottom-up chains after at most three scalar steps.
#pragma once
#include "afs_internal.h"

namespace afs {

__device__ __forceinline__ void load4(const float* p, float (&v)[4])
{
    float4 t = *reinterpret_cast<const float4*>(p);
    v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
}
__device__ __forceinline__ void load4(const double* p, double (&v)[4])
{
    double2 a = *reinterpret_cast<const double2*>(p), b = *reinterpret_cast<const double2*>(p + 2);
    v[0] = a.x; v[1] = a.y; v[2] = b.x; v[3] = b.y;
}
__device__ __forceinline__ float recip(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double recip(double x) { return 1.0 / x; }

// one literal, q_t += R q_{t-1}, on the live rows 0..PH
template <typename real, int NR, int PH>
__device__ __forceinline__ void dp_step(real (&q)[NR][4], const real R, const int lane)
{
    const int src = (lane + 31) & 31;
    real rot[PH + 1];
#pragma unroll
    for (int r = 0; r <= PH; ++r) rot[r] = __shfl_sync(0xffffffffu, q[r][3], src);
#pragma unroll
    for (int r = PH; r >= 0; --r) {
        real carry = rot[r];
        if (lane == 0) carry = r > 0 ? rot[r > 0 ? r - 1 : 0] : real(0);
        q[r][3] = fma(R, q[r][2], q[r][3]);
        q[r][2] = fma(R, q[r][1], q[r][2]);
        q[r][1] = fma(R, q[r][0], q[r][1]);
        q[r][0] = fma(R, carry, q[r][0]);
    }
}

// steps [s0, s1) with rows 0..PH live; s0 and s1 are multiples of 4
template <typename real, int NR, int PH>
__device__ __forceinline__ void dp_segment(real (&q)[NR][4], const real* __restrict__ Rc, int s0, int s1, int lane,
                                           real& P)
{
#pragma unroll 1
    for (int s = s0; s < s1; s += 4) {
        real R[4];
        load4(Rc + s, R);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            P = fma(P, R[e], P);
            dp_step<real, NR, PH>(q, R[e], lane);
        }
        if (((s + 4) & 31) == 0) {
            const real sc = recip(P);
#pragma unroll
            for (int r = 0; r <= PH; ++r)
#pragma unroll
                for (int i = 0; i < 4; ++i) q[r][i] *= sc;
            P = real(1);
        }
    }
}

template <typename real, int NR, int PH>
struct DpPhases {
    // steps [s0, s1) of the list
    static __device__ __forceinline__ void run(real (&q)[NR][4], const real* __restrict__ Rc, int s0, int s1, int lane,
                                               real& P)
    {
        if constexpr (PH < NR) {
            // rows 0..PH hold cells 0 .. 128(PH+1)-1; a group of four steps starting at s raises the degree to at most
            // s+4, so it may run in this phase while s + 4 <= 128(PH+1) - 1, i.e. (s a multiple of 4) s < 128(PH+1) - 4.
            // The last phase holds every cell up to L and takes everything that is left.
            const int lo = max(s0, PH == 0 ? 0 : 128 * PH - 4);
            const int hi = PH == NR - 1 ? s1 : min(s1, 128 * (PH + 1) - 4);
            if (lo < hi) dp_segment<real, NR, PH>(q, Rc, lo, hi, lane, P);
            DpPhases<real, NR, PH + 1>::run(q, Rc, s0, s1, lane, P);
        }
    }
};

// advance U chains s <- q_i - R s from chain index i through `target` inclusive.  Bottom-up (REV = false): q_i =
// A0[i]; top-down (REV = true): q_i = A0[-i].  mis = misalignment of A0 in elements (bottom-up only).
template <typename real, int U, bool REV>
__device__ __forceinline__ void chain_advance(const real* __restrict__ A0, int& i, int target, real (&s)[U],
                                              const real (&R)[U], int mis)
{
    while (i <= target && ((i + mis) & 3)) {
        const real v = REV ? A0[-i] : A0[i];
#pragma unroll
        for (int u = 0; u < U; ++u) s[u] = fma(-R[u], s[u], v);
        ++i;
    }
    int nblk = (target + 1 - i) >> 2;
    if (nblk > 0) {
        const real* p = REV ? A0 - i - 3 : A0 + i;
        i += nblk * 4;
#pragma unroll 1
        for (; nblk >= 2; nblk -= 2) {
            real v[4], w[4];
            load4(p, v);
            load4(REV ? p - 4 : p + 4, w);
            p = REV ? p - 8 : p + 8;
#pragma unroll
            for (int e = 0; e < 4; ++e)
#pragma unroll
                for (int u = 0; u < U; ++u) s[u] = fma(-R[u], s[u], REV ? v[3 - e] : v[e]);
#pragma unroll
            for (int e = 0; e < 4; ++e)
#pragma unroll
                for (int u = 0; u < U; ++u) s[u] = fma(-R[u], s[u], REV ? w[3 - e] : w[e]);
        }
        if (nblk) {
            real v[4];
            load4(p, v);
#pragma unroll
            for (int e = 0; e < 4; ++e)
#pragma unroll
                for (int u = 0; u < U; ++u) s[u] = fma(-R[u], s[u], REV ? v[3 - e] : v[e]);
        }
    }
    for (; i <= target; ++i) {
        const real v = REV ? A0[-i] : A0[i];
#pragma unroll
        for (int u = 0; u < U; ++u) s[u] = fma(-R[u], s[u], v);
    }
}

// one round of up to 32*U interior literals of one direction: list entries [0, cnt)
template <typename real, int U, bool REV>
__device__ __forceinline__ void deconv_round(const real* __restrict__ A0, int mis, real* __restrict__ Rc, int cnt,
                                             int c1, int c2, real w1, real w2, int lane)
{
    real R[U], s[U], s1[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int e = u * 32 + lane;
        R[u] = e < cnt ? Rc[e] : real(0);
        s[u] = real(0);
    }
    int i = 0;
    chain_advance<real, U, REV>(A0, i, c1, s, R, mis);
#pragma unroll
    for (int u = 0; u < U; ++u) s1[u] = s[u];
    chain_advance<real, U, REV>(A0, i, c2, s, R, mis);
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int e = u * 32 + lane;
        if (e < cnt) Rc[e] = (w1 * s1[u] + w2 * s[u]) * (real(1) + R[u]);   // dFE/dy_j replaces the ratio
    }
}

template <typename real, bool REV>
__device__ __forceinline__ void deconv_dir(const real* __restrict__ A0, int mis, real* __restrict__ Rc, int cnt, int c1,
                                           int c2, real w1, real w2, int lane)
{
#define AFS_ROUND(UU) deconv_round<real, UU, REV>(A0, mis, Rc + e0, rem, c1, c2, w1, w2, lane)
    for (int e0 = 0; e0 < cnt;) {
        const int rem = cnt - e0;
        if (rem > 96) { AFS_ROUND(4); e0 += 128; }
        else if (rem > 64) { AFS_ROUND(3); e0 += 96; }
        else if (rem > 32) { AFS_ROUND(2); e0 += 64; }
        else { AFS_ROUND(1); e0 += 32; }
    }
#undef AFS_ROUND
}

__device__ __forceinline__ bool long_pred(int type, int L, int k, int t)
{
    switch (type) {
    case AFS_OR: return t >= 1;
    case AFS_XOR: return ((t ^ k) & 1) == 0;
    case AFS_AMO: return t <= 1;
    case AFS_EO: return t == 1;
    case AFS_EK: return t == k;
    case AFS_NAE: return t > 0 && t < L;
    case AFS_CARD: return t >= k;
    default: return false;
    }
}

// One CTA = one constraint x one tile of 32 restarts; its RPC warps take the restarts of the tile in turn (warp w:
// restarts w, w + RPC, ...), each with its own list / pmf buffers.
//   words    the CTA first stages, per literal, the tile's "true" word (sign word of the variable, flipped for a negated
//            literal) and "saturated" word (|x| = 1) -- two 4-byte loads per literal for 32 restarts instead of 32
//            element gathers.  Bit r of the words classifies literal j for restart r: boundary-true, boundary-false,
//            interior with y < 0 (type B), interior with y >= 0 (type A).
//   pass 1   per restart, ballots over the words: true count tc (S9), boundary-true count nB0, nBr, nAr.  A restart
//            with no interior literal is finished here: its pmf is the point mass at nB0, the objective is -+1 and the
//            two boundary gradients are d_t picked at nB0 (no list, no gather, no arithmetic).
//   pass 2   otherwise: list positions from the same ballots, x gathered for the INTERIOR literals only.
//   output   boundary literals: ONE pair (dFE/dy at y = +1, at y = -1) per (constraint, restart) in bnd[c][b][2]; the
//            variable pass picks by its own x (a variable on +-1 is a boundary literal in every constraint it occurs
//            in).  Interior literals: their own scratch rows, as the other materialising classes.
template <typename real, int NR, int RPC>
__global__ void __launch_bounds__(RPC * 32) k_long(const LongCon* __restrict__ cons, int c_begin,
                                                   const uint32_t* __restrict__ lits, const int32_t* __restrict__ slots,
                                                   const real* __restrict__ XT, const uint32_t* __restrict__ Sw,
                                                   const uint32_t* __restrict__ SATw, int ntile, int Bp,
                                                   real* __restrict__ scratch, real* __restrict__ bnd,
                                                   int32_t* __restrict__ sat, real* __restrict__ fe_out, int LS, int QS,
                                                   unsigned long long* __restrict__ work)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    real* RcAll = reinterpret_cast<real*>(smem_raw);              // [RPC][LS]  ratios in list order, then gradients
    real* AAll = RcAll + RPC * LS;                                // [RPC][QS]  the pmf
    uint32_t* TW = reinterpret_cast<uint32_t*>(AAll + RPC * QS);  // [LS] true words of the tile
    uint32_t* SW = TW + LS;                                       // [LS] saturated words
    uint16_t* JAll = reinterpret_cast<uint16_t*>(SW + LS);        // [RPC][LS]  literal index at each list position
    constexpr int NT = RPC * 32;
    constexpr unsigned FULLM = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int c = c_begin + (int)(blockIdx.x / (unsigned)ntile);
    const int tile = (int)(blockIdx.x % (unsigned)ntile);
    const LongCon lc = cons[c];
    const int L = lc.L;
    const uint32_t* lw = lits + lc.off;
    const int32_t* sw = slots + lc.off;
    for (int j = tid; j < L; j += NT) {
        const uint32_t w = lw[j];
        const size_t wi = (size_t)(w & LIT_VAR) * ntile + tile;
        const uint32_t s = Sw[wi];
        TW[j] = (w >> 31) ? ~s : s;
        SW[j] = SATw[wi];
    }
    __syncthreads();
    real* Rc = RcAll + warp * LS;
    real* Aw = AAll + warp * QS;
    uint16_t* J = JAll + warp * LS;
    const bool useA = lc.wA != 0.f, useB = lc.wB != 0.f;
    // capture points in true-count index space, t1 <= t2 (equal if only one is used)
    int t1 = lc.tA, t2 = lc.tB;
    real w1 = (real)lc.wA, w2 = (real)lc.wB;
    if (!useA) { t1 = t2; w1 = real(0); }
    if (!useB) { t2 = t1; w2 = w1; w1 = real(0); }
    if (t1 > t2) { int tt = t1; t1 = t2; t2 = tt; real ww = w1; w1 = w2; w2 = ww; }
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll 1
    for (int r = warp; r < 32; r += RPC) {
        const int b = tile * 32 + r;
        // ---- pass 1: counts of the four literal kinds from the words
        int tc = 0, nB0 = 0, nBr = 0, nAr = 0;
        for (int j0 = 0; j0 < L; j0 += 32) {
            const int j = j0 + lane;
            const bool act = j < L;
            const bool tb = act && ((TW[act ? j : 0] >> r) & 1u), sb = !act || ((SW[act ? j : 0] >> r) & 1u);
            const unsigned mT = __ballot_sync(FULLM, tb), mS = __ballot_sync(FULLM, sb);
            const unsigned mAct = L - j0 >= 32 ? FULLM : (1u << (L - j0)) - 1u;
            tc += __popc(mT); nB0 += __popc(mT & mS); nBr += __popc(mT & ~mS); nAr += __popc(~mT & ~mS & mAct);
        }
        const int Leff = nBr + nAr;
        if (lane == 0 && sat && long_pred(lc.type, L, lc.k, tc)) atomicAdd(&sat[b], 1);
        auto dpick = [&](int tau) -> real {   // w1 [t1 = tau] + w2 [t2 = tau]: d_t at the point mass
            return (tau == t1 - nB0 ? w1 : real(0)) + (tau == t2 - nB0 ? w2 : real(0));
        };
        if (Leff == 0) {
            // every literal on the boundary: Q(z) = z^nB0.  Removing a false literal leaves the mass at nB0, removing a
            // true one moves it to nB0 - 1 (P:L52 d_t; exact, no arithmetic)
            if (lane == 0) {
                bnd[((size_t)c * Bp + b) * 2] = dpick(0);
                bnd[((size_t)c * Bp + b) * 2 + 1] = dpick(-1);
                if (fe_out) fe_out[(size_t)c * Bp + b] = long_pred(lc.type, L, lc.k, nB0) ? real(-1) : real(1);
            }
            continue;
        }
        // ---- pass 2: lists [B interior, pad | A interior, pad] of literal indices; x gathered for these only
        const int nBr4 = (nBr + 3) & ~3, nAr4 = (nAr + 3) & ~3, send = nBr4 + nAr4;
        {
            int pBr = 0, pAr = nBr4;
            for (int j0 = 0; j0 < L; j0 += 32) {
                const int j = j0 + lane;
                const bool act = j < L;
                const bool tb = act && ((TW[act ? j : 0] >> r) & 1u), intr = act && !((SW[act ? j : 0] >> r) & 1u);
                const bool cBr = intr && tb, cAr = intr && !tb;
                const unsigned mBr = __ballot_sync(FULLM, cBr), mAr = __ballot_sync(FULLM, cAr);
                if (intr) J[cBr ? pBr + __popc(mBr & lt) : pAr + __popc(mAr & lt)] = (uint16_t)j;
                pBr += __popc(mBr); pAr += __popc(mAr);
            }
            if (lane < nBr4 - nBr) J[nBr + lane] = 0xffffu;
            if (lane < nAr4 - nAr) J[nBr4 + nAr + lane] = 0xffffu;
        }
        __syncwarp();
        for (int e = lane; e < send; e += 32) {
            const int j = J[e];
            real R = real(0);   // neutral pad entry
            if (j != 0xffff) {
                const uint32_t w = lw[j];
                const real x = XT[(size_t)(w & LIT_VAR) * Bp + b];
                const real y = (w >> 31) ? -x : x;
                const real u = real(0.5) + real(0.5) * y, p = real(0.5) - real(0.5) * y;
                // the list decides the direction (type B: literal true by sign, p >= 1/2): min / max, divisor >= 1/2.
                // Correctly rounded reciprocal times the numerator (<= 1 ulp off the IEEE quotient)
                R = e < nBr4 ? u * recip(p) : p * recip(u);
            }
            Rc[e] = R;
        }
        // ---- S2: forward pmf of the interior literals
        const int off = (3 - Leff) & 3;
        {
            real q[NR][4];
#pragma unroll
            for (int rr = 0; rr < NR; ++rr)
#pragma unroll
                for (int i = 0; i < 4; ++i) q[rr][i] = real(0);
            if (lane == 0) q[0][0] = real(1);
            real P = real(1);
            for (int t = lane; t < QS; t += 32) Aw[t] = real(0);
            __syncwarp();
            if (nBr > 0) {
                DpPhases<real, NR, 0>::run(q, Rc, 0, nBr4, lane, P);
                // prod_B (z + R_j) is the reversal of prod_B (1 + R_j w): c_t -> c_{nBr - t}, through shared memory
#pragma unroll
                for (int rr = 0; rr < NR; ++rr)
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        int t = (rr * 32 + lane) * 4 + i;
                        if (t <= nBr) Aw[t] = q[rr][i];
                    }
                __syncwarp();
#pragma unroll
                for (int rr = 0; rr < NR; ++rr)
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        int t = (rr * 32 + lane) * 4 + i;
                        q[rr][i] = t <= nBr ? Aw[nBr - t] : real(0);
                    }
                __syncwarp();
                for (int t = lane; t <= nBr; t += 32) Aw[t] = real(0);
                __syncwarp();
            }
            DpPhases<real, NR, 0>::run(q, Rc, nBr4, send, lane, P);
            const real sc = recip(P);
            real fe = real(0);
#pragma unroll
            for (int rr = 0; rr < NR; ++rr)
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    int t = (rr * 32 + lane) * 4 + i;
                    if (t <= Leff) {
                        const real v = q[rr][i] * sc;
                        Aw[off + t] = v;
                        fe += long_pred(lc.type, L, lc.k, t + nB0) ? -v : v;   // sp = -1 where satisfied
                    }
                }
            if (fe_out) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) fe += __shfl_xor_sync(FULLM, fe, o);
                if (lane == 0) fe_out[(size_t)c * Bp + b] = fe;
            }
        }
        __syncwarp();
        // ---- S3 + S5: leave-one-out
        // timing mode only: the state-dependent algorithmic work of this (constraint, restart) -- 6 Leff Keff flops, the
        // survey's count for a pmf of Leff interior literals with the threshold left after the nB0 true boundary literals
        if (work && lane == 0) {
            const int keff = lc.k - nB0;
            const bool live = (useA || useB) && keff >= (lc.type == AFS_EK ? 0 : 1) && keff <= Leff;
            if (live) {
                int K = min(keff, Leff - keff + 1) + 1;
                K = K < 1 ? 1 : K;
                atomicAdd(work + (blockIdx.x & 31u), 6ull * (unsigned long long)Leff * (unsigned long long)K);   // 32 slots
            }
        }
        const real* qr = Aw + off;   // qr[tau] = reduced pmf, tau in [0, Leff]; q_t = qr[t - nB0]
        // boundary literals: y = +1 leaves q unchanged, y = -1 removes one shift (q^(-j)_t = q_{t+1})
        if (lane == 0) {
            auto qat = [&](int tau) -> real { return (tau >= 0 && tau <= Leff) ? qr[tau] : real(0); };
            bnd[((size_t)c * Bp + b) * 2] = w1 * qat(t1 - nB0) + w2 * qat(t2 - nB0);
            bnd[((size_t)c * Bp + b) * 2 + 1] = w1 * qat(t1 + 1 - nB0) + w2 * qat(t2 + 1 - nB0);
        }
        // interior literals: q^(-j)_t = qred^(-j)_{t - nB0}, qred^(-j) has degree Leff - 1
        int c1 = t1 - nB0, c2 = t2 - nB0;
        real v1w = w1, v2w = w2;
        const bool v1 = c1 >= 0 && c1 <= Leff - 1 && w1 != real(0), v2 = c2 >= 0 && c2 <= Leff - 1 && w2 != real(0);
        if (!v1 && !v2) {   // the expansion does not depend on the interior literals here (or is constant): zero gradient
            for (int e = lane; e < send; e += 32) Rc[e] = real(0);
        } else {
            if (!v1) { c1 = c2; v1w = real(0); }
            if (!v2) { c2 = c1; v2w = v1w; v1w = real(0); }
            // type A: bottom-up chain over qr_0, qr_1, ...; captures at c1 then c2
            deconv_dir<real, false>(qr, off, Rc + nBr4, nAr, c1, c2, v1w, v2w, lane);
            // type B: top-down chain over qr_Leff, qr_{Leff-1}, ...; chain index i <-> tau = Leff-1-i, so c2 is met first
            deconv_dir<real, true>(qr + Leff, 0, Rc, nBr, Leff - 1 - c2, Leff - 1 - c1, v2w, v1w, lane);
        }
        __syncwarp();
        // ---- S5 + write-out of the interior literals' rows
        for (int e = lane; e < send; e += 32) {
            const int j = J[e];
            if (j != 0xffff) {
                const real g = Rc[e];
                scratch[(size_t)sw[j] * Bp + b] = (lw[j] >> 31) ? -g : g;
            }
        }
        __syncwarp();
    }
}

}  // namespace afs
