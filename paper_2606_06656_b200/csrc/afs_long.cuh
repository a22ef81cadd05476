// afs_long.cuh -- the LONG class: EK / CARD longer than 64 literals (and NAE / EO / AMO too long for the register
// kernels).  warp = (constraint, restart), CTA = one constraint x RPC restarts.  Count basis (G10):
//   gather    per literal the ratio R = min(u, p) / max(u, p) in [0, 1] and its direction (type A: p <= 1/2, type B:
//             p > 1/2); max(u, p) = 1 / (1 + R) because u + p = 1.  The literals of a restart are then compacted by
//             type (A first, padded with neutral R = 0 entries to a multiple of four, then B).
//   forward   Q(z) = prod_j (u_j + p_j z) = prod_A (1 + R_j z) * prod_B (z + R_j) / prod_j (1 + R_j): the pmf q of the
//             number of true literals is built with ONE FMA per cell and literal -- A: q_t += R q_{t-1};  B: q_t =
//             q_{t-1} + R q_t -- and the scalar 1 / prod (1 + R_j) is applied every 32 literals (growth inside a block
//             <= 2^32).  The pmf lives in registers, cell t = (row*32 + lane)*4 + c; rows that are still identically
//             zero are skipped (warp-uniform).
//   gradient  dFE/dy_j = sum_t d_t q_t^(-j) with at most two non-zero d_t.  q^(-j) comes from q by removing
//             literal j in the STABLE direction: s_t = q_t - R_j s_{t-1} from the bottom for type A, the same
//             recurrence from the top for type B; q^(-j) = (1 + R_j) s.  Nothing that vanishes at x = +-1 is ever
//             divided by (BASELINE.json subsystem (2)).  A warp runs chains of one direction and one length; every
//             lane carries up to four chains that share each broadcast load of q.
// The pmf sits in shared memory at A[off + t] with off = (3 - L) mod 4, so that the top-down chains read aligned
// 16-byte blocks from index 0 and the bottom-up chains after at most three scalar steps.
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

// one literal on the live rows 0..PH
template <typename real, int NR, int PH, bool TYPEB>
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
        if (!TYPEB) {
            q[r][3] = fma(R, q[r][2], q[r][3]);
            q[r][2] = fma(R, q[r][1], q[r][2]);
            q[r][1] = fma(R, q[r][0], q[r][1]);
            q[r][0] = fma(R, carry, q[r][0]);
        } else {
            q[r][3] = fma(R, q[r][3], q[r][2]);
            q[r][2] = fma(R, q[r][2], q[r][1]);
            q[r][1] = fma(R, q[r][1], q[r][0]);
            q[r][0] = fma(R, q[r][0], carry);
        }
    }
}

template <typename real, int NR, int PH>
__device__ __forceinline__ void dp_rescale(real (&q)[NR][4], real& P)
{
    const real sc = real(1) / P;
#pragma unroll
    for (int r = 0; r <= PH; ++r)
#pragma unroll
        for (int i = 0; i < 4; ++i) q[r][i] *= sc;
    P = real(1);
}

// steps [s0, s1) of one type with rows 0..PH live; s0 is a multiple of 4
template <typename real, int NR, int PH, bool TYPEB>
__device__ __forceinline__ void dp_segment(real (&q)[NR][4], const real* __restrict__ Rc, int s0, int s1, int lane,
                                           real& P)
{
    int s = s0;
    for (; s + 4 <= s1; s += 4) {
        real R[4];
        load4(Rc + s, R);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            P = fma(P, R[e], P);
            dp_step<real, NR, PH, TYPEB>(q, R[e], lane);
        }
        if (((s + 4) & 31) == 0) dp_rescale<real, NR, PH>(q, P);
    }
    for (; s < s1; ++s) {   // tail of the type-B section (at most three literals; no 32-boundary can fall inside)
        const real R = Rc[s];
        P = fma(P, R, P);
        dp_step<real, NR, PH, TYPEB>(q, R, lane);
    }
}

template <typename real, int NR, int PH>
struct DpPhases {
    // nA4: end of the (padded) type-A section, send: end of the type-B section
    static __device__ __forceinline__ void run(real (&q)[NR][4], const real* __restrict__ Rc, int nA4, int send, int lane,
                                               real& P)
    {
        if constexpr (PH < NR) {
            // rows 0..PH hold cells 0 .. 128(PH+1)-1; a group of four steps starting at s raises the degree to at most
            // s+4, so it may run in this phase while s + 4 <= 128(PH+1) - 1, i.e. (s a multiple of 4) s < 128(PH+1) - 4.
            // The last phase holds every cell up to L and takes everything that is left.
            const int lo = PH == 0 ? 0 : 128 * PH - 4;
            const int hi = PH == NR - 1 ? send + 4 : 128 * (PH + 1) - 4;
            if (lo < send) {
                const int a1 = min(hi, nA4);
                if (lo < a1) dp_segment<real, NR, PH, false>(q, Rc, lo, a1, lane, P);
                const int b0 = max(lo, nA4), b1 = min(hi, send);
                if (b0 < b1) dp_segment<real, NR, PH, true>(q, Rc, b0, b1, lane, P);
            }
            DpPhases<real, NR, PH + 1>::run(q, Rc, nA4, send, lane, P);
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
    for (; i + 3 <= target; i += 4) {
        real v[4];
        if (REV) load4(A0 - i - 3, v); else load4(A0 + i, v);
#pragma unroll
        for (int e = 0; e < 4; ++e)
#pragma unroll
            for (int u = 0; u < U; ++u) s[u] = fma(-R[u], s[u], REV ? v[3 - e] : v[e]);
    }
    for (; i <= target; ++i) {
        const real v = REV ? A0[-i] : A0[i];
#pragma unroll
        for (int u = 0; u < U; ++u) s[u] = fma(-R[u], s[u], v);
    }
}

// one round of up to 32*U literals of one direction: list entries [0, cnt)
template <typename real, int U, bool REV>
__device__ __forceinline__ void deconv_round(const real* __restrict__ A0, int mis, const uint16_t* __restrict__ lst,
                                             const real* __restrict__ Rc, int cnt, int c1, int c2, real w1, real w2,
                                             const uint32_t* __restrict__ lw, const int32_t* __restrict__ sw,
                                             real* __restrict__ scratch, size_t Bp, int b, int lane)
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
        if (e < cnt) {
            const int j = (int)lst[e];
            const real g = (w1 * s1[u] + w2 * s[u]) * (real(1) + R[u]);
            const uint32_t w = lw[j];
            scratch[(size_t)sw[j] * Bp + b] = (w >> 31) ? -g : g;
        }
    }
}

template <typename real, bool REV>
__device__ __forceinline__ void deconv_dir(const real* __restrict__ A0, int mis, const uint16_t* __restrict__ lst,
                                           const real* __restrict__ Rc, int cnt, int c1, int c2, real w1, real w2,
                                           const uint32_t* __restrict__ lw, const int32_t* __restrict__ sw,
                                           real* __restrict__ scratch, size_t Bp, int b, int lane)
{
#define AFS_ROUND(UU) \
    deconv_round<real, UU, REV>(A0, mis, lst + e0, Rc + e0, rem, c1, c2, w1, w2, lw, sw, scratch, Bp, b, lane)
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
                                                   int32_t* __restrict__ sat, real* __restrict__ fe_out, int LS, int QS)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    real* RcAll = reinterpret_cast<real*>(smem_raw);              // [RPC][LS]  ratios in list order
    real* AAll = RcAll + RPC * LS;                                // [RPC][QS]  signed ratios (gather), then the pmf
    uint16_t* LstAll = reinterpret_cast<uint16_t*>(AAll + RPC * QS);   // [RPC][LS]  literal index of each list entry
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
        for (int idx = tid; idx < ((L * RPC + NT - 1) / NT) * NT; idx += NT) {
            int j = idx / RPC;
            bool tr = false;
            if (j < L) {
                uint32_t w = lw[j];
                real x = XT[(size_t)(w & LIT_VAR) * Bp + bg * RPC + r];
                bool neg = (w >> 31) != 0;
                tr = (x < real(0)) != neg;
                const real y = neg ? -x : x;
                const real u = real(0.5) + real(0.5) * y, p = real(0.5) - real(0.5) * y;
                const bool fwd = !(y < real(0));             // p <= 1/2: type A
                const real R = fwd ? p / u : u / p;          // in [0, 1]; the divisor is >= 1/2
                AAll[r * QS + j] = fwd ? R : -R;             // -0.0 keeps the direction when R = 0
            }
            unsigned bal = __ballot_sync(FULLM, tr);
            if (lane < RPC) {
                int add = __popc(bal & (pat << lane));
                if (add) atomicAdd(&s_cnt[lane], add);
            }
        }
    }
    __syncthreads();
    const int b = bg * RPC + warp;
    real* Rc = RcAll + warp * LS;
    real* Aw = AAll + warp * QS;
    uint16_t* lst = LstAll + warp * LS;
    // ---- compaction by direction: A entries [0, nA), zeros up to nA4, B entries [nA4, nA4 + nB)
    int nA = 0;
    for (int j0 = 0; j0 < L; j0 += 32) {
        const int j = j0 + lane;
        nA += __popc(__ballot_sync(FULLM, j < L && !signbit(Aw[j < L ? j : 0])));
    }
    const int nA4 = (nA + 3) & ~3, nB = L - nA, send = nA4 + nB;
    {
        const unsigned lt = (1u << lane) - 1u;
        int pa = 0, pb = nA4;
        for (int j0 = 0; j0 < L; j0 += 32) {
            const int j = j0 + lane;
            const bool act = j < L;
            const real rs = Aw[act ? j : 0];
            const bool isB = act && signbit(rs);
            const bool isA = act && !isB;
            const unsigned bA = __ballot_sync(FULLM, isA), bB = __ballot_sync(FULLM, isB);
            const int pos = isA ? pa + __popc(bA & lt) : pb + __popc(bB & lt);
            if (act) { Rc[pos] = fabs(rs); lst[pos] = (uint16_t)j; }
            pa += __popc(bA); pb += __popc(bB);
        }
        if (lane < nA4 - nA) Rc[nA + lane] = real(0);
    }
    __syncwarp();
    // ---- S2: forward pmf
    const int off = (3 - L) & 3;
    {
        real q[NR][4];
#pragma unroll
        for (int r = 0; r < NR; ++r)
#pragma unroll
            for (int i = 0; i < 4; ++i) q[r][i] = real(0);
        if (lane == 0) q[0][0] = real(1);
        real P = real(1);
        DpPhases<real, NR, 0>::run(q, Rc, nA4, send, lane, P);
        const real sc = real(1) / P;
        real fe = real(0);
        for (int t = lane; t < QS; t += 32) Aw[t] = real(0);   // the signed ratios are no longer needed
        __syncwarp();
#pragma unroll
        for (int r = 0; r < NR; ++r)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                int t = (r * 32 + lane) * 4 + i;
                if (t <= L) {
                    const real v = q[r][i] * sc;
                    Aw[off + t] = v;
                    fe += long_pred(lc.type, L, lc.k, t) ? -v : v;   // sp_t = -1 where satisfied
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
    // ---- S3 + S5: leave-one-out by stable-direction deconvolution
    const bool useA = lc.wA != 0.f, useB = lc.wB != 0.f;
    if (!useA && !useB) {   // constant expansion (CARD with k = 0 or k = L+1): zero gradient
        for (int j = lane; j < L; j += 32) scratch[(size_t)sw[j] * Bp + b] = real(0);
        return;
    }
    // capture points in true-count index space, t1 <= t2 (equal if only one is used)
    int t1 = lc.tA, t2 = lc.tB;
    real w1 = (real)lc.wA, w2 = (real)lc.wB;
    if (!useA) { t1 = t2; w1 = real(0); }
    if (!useB) { t2 = t1; w2 = w1; w1 = real(0); }
    if (t1 > t2) { int tt = t1; t1 = t2; t2 = tt; real ww = w1; w1 = w2; w2 = ww; }
    // type A: bottom-up chain over q_0, q_1, ...; captures at t1 then t2
    deconv_dir<real, false>(Aw + off, off, lst, Rc, nA, t1, t2, w1, w2, lw, sw, scratch, (size_t)Bp, b, lane);
    // type B: top-down chain over q_L, q_{L-1}, ...; chain index i <-> t = L-1-i, so t2 is met first
    deconv_dir<real, true>(Aw + off + L, 0, lst + nA4, Rc + nA4, nB, L - 1 - t2, L - 1 - t1, w2, w1, lw, sw, scratch,
                           (size_t)Bp, b, lane);
}

}  // namespace afs
