// afs_long.cuh -- the LONG class: EK / CARD longer than 64 literals (and NAE / EO / AMO too long for the register
// kernels).  warp = (constraint, restart), CTA = one constraint x RPC restarts.  Count basis (G10):
//
//   Q(z) = prod_j (u_j + p_j z),  u = (1+y)/2, p = (1-y)/2,  q_t = [z^t] Q = Pr[t literals true]
//
//   gather    per literal the ratio R = min(u, p) / max(u, p) in [0, 1] and its direction (type A: p <= 1/2, type B:
//             p > 1/2); max(u, p) = 1 / (1 + R) because u + p = 1.  A literal on the boundary of the cube has R = 0:
//             y = +1 is the factor 1, y = -1 is the factor z -- an exact shift of the pmf, no arithmetic.  PGD iterates
//             sit on that boundary in most coordinates (clipping; fixed variables), so the pmf is
//             built from the INTERIOR literals only:  Q(z) = z^nB0 * Qred(z),  deg Qred = Leff.
//   lists     the literals of a restart are compacted into  [ B interior | A interior | A boundary | B boundary ],
//             the interior sections padded with neutral R = 0 entries to multiples of four.
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
//             q^(-j) = q (y = +1) or q shifted by one (y = -1).
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

template <typename real, int NR, int RPC>
__global__ void __launch_bounds__(RPC * 32) k_long(const LongCon* __restrict__ cons, int c_begin,
                                                   const uint32_t* __restrict__ lits, const int32_t* __restrict__ slots,
                                                   const real* __restrict__ XT, int Bp, real* __restrict__ scratch,
                                                   int32_t* __restrict__ sat, real* __restrict__ fe_out, int LS, int QS,
                                                   unsigned long long* __restrict__ work)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    real* RcAll = reinterpret_cast<real*>(smem_raw);              // [RPC][LS]  ratios in list order
    real* AAll = RcAll + RPC * LS;                                // [RPC][QS]  signed ratios (gather), then the pmf
    uint16_t* InvAll = reinterpret_cast<uint16_t*>(AAll + RPC * QS);   // [RPC][LS]  list position of each literal
    __shared__ int s_cnt[RPC];
    constexpr int NT = RPC * 32;
    constexpr unsigned FULLM = 0xffffffffu;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int groups = Bp / RPC;
    const int c = c_begin + (int)(blockIdx.x / groups);
    const int bg = (int)(blockIdx.x % groups);
    const LongCon lc = cons[c];
    const int L = lc.L;
    const uint32_t* lw = lits + lc.off;
    const int32_t* sw = slots + lc.off;
    if (tid < RPC) s_cnt[tid] = 0;
    __syncthreads();
    // ---- S1: gather the literal values of RPC consecutive restarts (one 32-byte sector per literal for 8 x fp32)
    {
        const int r = tid % RPC;
        const unsigned pat = RPC == 8 ? 0x01010101u : RPC == 4 ? 0x11111111u : RPC == 2 ? 0x55555555u : 0xffffffffu;
        // four rounds of the block at a time: the literal words first, then the four gathers, so that a thread has four
        // dependent (word -> row) pairs in flight instead of one
        const int rounds = (L * RPC + NT - 1) / NT;
        int truec = 0;   // lanes < RPC: true literals of restart `lane` seen by this warp
        for (int r0 = 0; r0 < rounds; r0 += 4) {
            uint32_t w[4];
            real x[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int j = (tid + (r0 + k) * NT) / RPC;
                w[k] = j < L ? lw[j] : 0u;
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const int j = (tid + (r0 + k) * NT) / RPC;
                x[k] = j < L ? XT[(size_t)(w[k] & LIT_VAR) * Bp + bg * RPC + r] : real(0);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                if (r0 + k < rounds) {   // block-uniform
                    const int j = (tid + (r0 + k) * NT) / RPC;
                    bool tr = false;
                    if (j < L) {
                        const bool neg = (w[k] >> 31) != 0;
                        tr = (x[k] < real(0)) != neg;
                        const real y = neg ? -x[k] : x[k];
                        const real u = real(0.5) + real(0.5) * y, p = real(0.5) - real(0.5) * y;
                        const bool fwd = !(y < real(0));             // p <= 1/2: type A
                        // in [0, 1]; the divisor is >= 1/2; 0 on the boundary.  Correctly rounded reciprocal times the
                        // numerator (one MUFU + two corrections instead of the IEEE division sequence; <= 1 ulp off)
                        const real R = (fwd ? p : u) * recip(fwd ? u : p);
                        AAll[r * QS + j] = fwd ? R : -R;             // the sign bit is the direction (-0.0 for y = -1)
                    }
                    const unsigned bal = __ballot_sync(FULLM, tr);
                    if (lane < RPC) truec += __popc(bal & (pat << lane));
                }
            }
        }
        if (lane < RPC && truec) atomicAdd(&s_cnt[lane], truec);
    }
    __syncthreads();
    const int b = bg * RPC + warp;
    real* Rc = RcAll + warp * LS;
    real* Aw = AAll + warp * QS;
    uint16_t* inv = InvAll + warp * LS;
    // ---- lists: [B interior, pad | A interior, pad]; the boundary literals share two slots behind them (send: y = +1,
    // send + 1: y = -1), because all literals of one kind get the same gradient
    int nBr = 0, nAr = 0, nA0 = 0;
    for (int j0 = 0; j0 < L; j0 += 32) {
        const int j = j0 + lane;
        const bool act = j < L;
        const real rs = Aw[act ? j : 0];
        const bool isB = signbit(rs), intr = rs != real(0);
        nBr += __popc(__ballot_sync(FULLM, act && isB && intr));
        nAr += __popc(__ballot_sync(FULLM, act && !isB && intr));
        nA0 += __popc(__ballot_sync(FULLM, act && !isB && !intr));
    }
    const int nB0 = L - nBr - nAr - nA0;
    const int nBr4 = (nBr + 3) & ~3, nAr4 = (nAr + 3) & ~3, send = nBr4 + nAr4, Leff = nBr + nAr;
    {
        const unsigned lt = (1u << lane) - 1u;
        int pBr = 0, pAr = nBr4;
        for (int j0 = 0; j0 < L; j0 += 32) {
            const int j = j0 + lane;
            const bool act = j < L;
            const real rs = Aw[act ? j : 0];
            const bool isB = signbit(rs), intr = rs != real(0);
            const bool cBr = act && isB && intr, cAr = act && !isB && intr;
            const unsigned mBr = __ballot_sync(FULLM, cBr), mAr = __ballot_sync(FULLM, cAr);
            const int pos = cBr ? pBr + __popc(mBr & lt) : cAr ? pAr + __popc(mAr & lt) : send + (isB ? 1 : 0);
            if (act) {
                inv[j] = (uint16_t)pos;
                if (intr) Rc[pos] = fabs(rs);
            }
            pBr += __popc(mBr); pAr += __popc(mAr);
        }
        if (lane < nBr4 - nBr) Rc[nBr + lane] = real(0);
        if (lane < nAr4 - nAr) Rc[nBr4 + nAr + lane] = real(0);
    }
    __syncwarp();
    // ---- S2: forward pmf of the interior literals
    const int off = (3 - Leff) & 3;
    {
        real q[NR][4];
#pragma unroll
        for (int r = 0; r < NR; ++r)
#pragma unroll
            for (int i = 0; i < 4; ++i) q[r][i] = real(0);
        if (lane == 0) q[0][0] = real(1);
        real P = real(1);
        for (int t = lane; t < QS; t += 32) Aw[t] = real(0);   // the signed ratios are no longer needed
        __syncwarp();
        if (nBr > 0) {
            DpPhases<real, NR, 0>::run(q, Rc, 0, nBr4, lane, P);
            // prod_B (z + R_j) is the reversal of prod_B (1 + R_j w): c_t -> c_{nBr - t}, through shared memory
#pragma unroll
            for (int r = 0; r < NR; ++r)
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    int t = (r * 32 + lane) * 4 + i;
                    if (t <= nBr) Aw[t] = q[r][i];
                }
            __syncwarp();
#pragma unroll
            for (int r = 0; r < NR; ++r)
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    int t = (r * 32 + lane) * 4 + i;
                    q[r][i] = t <= nBr ? Aw[nBr - t] : real(0);
                }
            __syncwarp();
            for (int t = lane; t <= nBr; t += 32) Aw[t] = real(0);
            __syncwarp();
        }
        DpPhases<real, NR, 0>::run(q, Rc, nBr4, send, lane, P);
        const real sc = recip(P);
        real fe = real(0);
#pragma unroll
        for (int r = 0; r < NR; ++r)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                int t = (r * 32 + lane) * 4 + i;
                if (t <= Leff) {
                    const real v = q[r][i] * sc;
                    Aw[off + t] = v;
                    fe += long_pred(lc.type, L, lc.k, t + nB0) ? -v : v;   // sp = -1 where satisfied
                }
            }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) fe += __shfl_xor_sync(FULLM, fe, o);
        if (lane == 0) {
            if (fe_out) fe_out[(size_t)c * Bp + b] = fe;
            if (sat && long_pred(lc.type, L, lc.k, s_cnt[warp])) atomicAdd(&sat[b], 1);
        }
    }
    __syncwarp();
    // ---- S3 + S5: leave-one-out
    const bool useA = lc.wA != 0.f, useB = lc.wB != 0.f;
    // timing mode only: the state-dependent algorithmic work of this (constraint, restart) -- 6 Leff Keff flops, the
    // survey's count for a pmf of Leff interior literals with the threshold left after the nB0 true boundary literals
    if (work && lane == 0) {
        const int keff = lc.k - nB0;
        const bool live = (useA || useB) && Leff > 0 && keff >= (lc.type == AFS_EK ? 0 : 1) && keff <= Leff;
        if (live) {
            int K = min(keff, Leff - keff + 1) + 1;
            K = K < 1 ? 1 : K;
            atomicAdd(work + (blockIdx.x & 31u), 6ull * (unsigned long long)Leff * (unsigned long long)K);   // 32 slots
        }
    }
    // capture points in true-count index space, t1 <= t2 (equal if only one is used)
    int t1 = lc.tA, t2 = lc.tB;
    real w1 = (real)lc.wA, w2 = (real)lc.wB;
    if (!useA) { t1 = t2; w1 = real(0); }
    if (!useB) { t2 = t1; w2 = w1; w1 = real(0); }
    if (t1 > t2) { int tt = t1; t1 = t2; t2 = tt; real ww = w1; w1 = w2; w2 = ww; }
    const real* qr = Aw + off;   // qr[tau] = reduced pmf, tau in [0, Leff]; q_t = qr[t - nB0]
    // boundary literals: y = +1 leaves q unchanged, y = -1 removes one shift (q^(-j)_t = q_{t+1}).  Every dFE/dy_j
    // goes to Rc at the literal's list position; the CTA then writes whole 32-byte sectors of the scratch rows.
    {
        auto qat = [&](int tau) -> real { return (tau >= 0 && tau <= Leff) ? qr[tau] : real(0); };
        const real gA0 = w1 * qat(t1 - nB0) + w2 * qat(t2 - nB0);
        const real gB0 = w1 * qat(t1 + 1 - nB0) + w2 * qat(t2 + 1 - nB0);
        if (lane < 2) Rc[send + lane] = lane == 0 ? gA0 : gB0;
    }
    // interior literals: q^(-j)_t = qred^(-j)_{t - nB0}, qred^(-j) has degree Leff - 1
    int c1 = t1 - nB0, c2 = t2 - nB0;
    const bool v1 = c1 >= 0 && c1 <= Leff - 1 && w1 != real(0), v2 = c2 >= 0 && c2 <= Leff - 1 && w2 != real(0);
    if (!v1 && !v2) {   // the expansion does not depend on the interior literals here (or is constant): zero gradient
        for (int e = lane; e < send; e += 32) Rc[e] = real(0);
    } else {
        if (!v1) { c1 = c2; w1 = real(0); }
        if (!v2) { c2 = c1; w2 = w1; w1 = real(0); }
        // type A: bottom-up chain over qr_0, qr_1, ...; captures at c1 then c2
        deconv_dir<real, false>(qr, off, Rc + nBr4, nAr, c1, c2, w1, w2, lane);
        // type B: top-down chain over qr_Leff, qr_{Leff-1}, ...; chain index i <-> tau = Leff-1-i, so c2 is met first
        deconv_dir<real, true>(qr + Leff, 0, Rc, nBr, Leff - 1 - c2, Leff - 1 - c1, w2, w1, lane);
    }
    __syncthreads();
    // ---- S5 + write-out: thread = (literal, restart), restart fastest
    {
        const int r = tid % RPC;
        const real* Rr = RcAll + r * LS;
        const uint16_t* ir = InvAll + r * LS;
        real* dst = scratch + (size_t)bg * RPC + r;
#pragma unroll 4
        for (int idx = tid; idx < L * RPC; idx += NT) {
            const int j = idx / RPC;
            const real g = Rr[ir[j]];
            dst[(size_t)sw[j] * Bp] = (lw[j] >> 31) ? -g : g;
        }
    }
}

}  // namespace afs
