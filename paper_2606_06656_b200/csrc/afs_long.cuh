// afs_long.cuh -- the LONG class: EK / CARD longer than 64 literals (nothing else is ever sorted into it).
// Count basis (G10):
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
#include "afs_bits.cuh"
#include "afs_retire.cuh"

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

// Forward pmf of the interior literals of one restart (list ratios Rc[0, send), nBr of them type B), NRR rows of 128
// cells in registers; leaves the reduced pmf at Aw[off + t], t = 0..Leff, and returns this lane's share of
// FE = sum_t sp_t q_t (sp = -1 where the constraint holds with t + nB0 true literals).
template <typename real, int NRR>
__device__ __forceinline__ real long_forward(const LongCon& lc, const int L, real* __restrict__ Rc, real* __restrict__ Aw,
                                             const int nBr, const int nBr4, const int send, const int Leff, const int nB0,
                                             const int off, const int lane, const int QS, const bool want_fe)
{
    constexpr unsigned FULLM = 0xffffffffu;
    real q[NRR][4];
#pragma unroll
    for (int rr = 0; rr < NRR; ++rr)
#pragma unroll
        for (int i = 0; i < 4; ++i) q[rr][i] = real(0);
    if (lane == 0) q[0][0] = real(1);
    real P = real(1);
    for (int t = lane; t < min(QS, Leff + 12); t += 32) Aw[t] = real(0);   // cells the reversal, the pmf and the chains' blocks touch
    __syncwarp();
    if (nBr > 0) {
        DpPhases<real, NRR, 0>::run(q, Rc, 0, nBr4, lane, P);
        // prod_B (z + R_j) is the reversal of prod_B (1 + R_j w): c_t -> c_{nBr - t}, through shared memory
#pragma unroll
        for (int rr = 0; rr < NRR; ++rr)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                int t = (rr * 32 + lane) * 4 + i;
                if (t <= nBr) Aw[t] = q[rr][i];
            }
        __syncwarp();
#pragma unroll
        for (int rr = 0; rr < NRR; ++rr)
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                int t = (rr * 32 + lane) * 4 + i;
                q[rr][i] = t <= nBr ? Aw[nBr - t] : real(0);
            }
        __syncwarp();
        for (int t = lane; t <= nBr; t += 32) Aw[t] = real(0);
        __syncwarp();
    }
    DpPhases<real, NRR, 0>::run(q, Rc, nBr4, send, lane, P);
    const real sc = recip(P);
    real fe = real(0);
#pragma unroll
    for (int rr = 0; rr < NRR; ++rr)
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            int t = (rr * 32 + lane) * 4 + i;
            if (t <= Leff) {
                const real v = q[rr][i] * sc;
                Aw[off + t] = v;
                if (want_fe) fe += long_pred(lc.type, L, lc.k, t + nB0) ? -v : v;
            }
        }
    (void)FULLM;
    return fe;
}

// The same for Leff < 32 CPL: the whole pmf in CPL cells per lane (cell t = lane * CPL + i), CPL + 5 instructions per
// literal, no rows to manage.  No rescaling on the way: the un-normalised coefficients grow by at most 2 per literal
// (R <= 1), 2^120 in all, inside the fp32 range.
template <typename real, int CPL>
__device__ __forceinline__ real long_forward_small(const LongCon& lc, const int L, const real* __restrict__ Rc,
                                                   real* __restrict__ Aw, const int nBr, const int nBr4, const int nAr,
                                                   const int Leff, const int nB0, const int off, const int lane,
                                                   const int QS, const bool want_fe)
{
    constexpr unsigned FULLM = 0xffffffffu;
    real q[CPL];
#pragma unroll
    for (int i = 0; i < CPL; ++i) q[i] = real(0);
    if (lane == 0) q[0] = real(1);
    real P = real(1);
    auto step = [&](const real R) {
        real lo = __shfl_up_sync(FULLM, q[CPL - 1], 1);
        if (lane == 0) lo = real(0);
#pragma unroll
        for (int i = CPL - 1; i >= 1; --i) q[i] = fma(R, q[i - 1], q[i]);
        q[0] = fma(R, lo, q[0]);
        P = fma(P, R, P);
    };
    for (int e = 0; e < nBr; ++e) step(Rc[e]);
    if (nBr > 0) {   // prod_B (z + R_j) is the reversal of prod_B (1 + R_j w): c_t -> c_{nBr - t}, through shared memory
#pragma unroll
        for (int i = 0; i < CPL; ++i) { const int t = lane * CPL + i; if (t <= nBr) Aw[t] = q[i]; }
        __syncwarp();
#pragma unroll
        for (int i = 0; i < CPL; ++i) { const int t = lane * CPL + i; q[i] = t <= nBr ? Aw[nBr - t] : real(0); }
        __syncwarp();
    }
    for (int e = 0; e < nAr; ++e) step(Rc[nBr4 + e]);
    const real sc = recip(P);
    for (int t = lane; t < min(QS, Leff + 12); t += 32) Aw[t] = real(0);   // cells the chains' 16-byte blocks touch
    __syncwarp();
    real fe = real(0);
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const int t = lane * CPL + i;
        if (t <= Leff) {
            const real v = q[i] * sc;
            Aw[off + t] = v;
            if (want_fe) fe += long_pred(lc.type, L, lc.k, t + nB0) ? -v : v;
        }
    }
    return fe;
}

// Two kernels per PGD iteration.
//
// k_long_scan   warp = (constraint, tile of 32 restarts).  Lane <-> literal: the tile's "true" word (sign word of the
//               variable, flipped for a negated literal) and "saturated" word (|x| = 1) of 32 literals at a time -- two
//               4-byte loads per literal for 32 restarts instead of 32 element gathers -- give three 32 x 32 bit
//               matrices (boundary-true, interior-true = type B, interior-false = type A) whose column sums (butterfly,
//               lane r <-> restart r afterwards) are nB0, nBr, nAr of every restart.  Then, lane <-> restart:
//                 S9   the constraint holds for nB0 + nBr true literals -> integer add to sat[b];
//                 Leff = nBr + nAr = 0 (every literal on the boundary): Q(z) = z^nB0, the objective is -+1 and the two
//                      boundary gradients are d_t picked at nB0 -- finished here, no list, no gather, no
//                      arithmetic;
//                 otherwise the pair (constraint, restart) is appended to the work list of its size class (rows of 128
//                      pmf cells that Leff needs); the order of a list does not enter any result.
// k_long_items  warp = one work-list entry.  Interior literals found from the same words (one restart's bits), x gathered
//               for these only, forward pmf, leave-one-out chains.
// Output of both: boundary literals get ONE pair (dFE/dy at y = +1, at y = -1) per (constraint, restart) in
// bnd[c][b][2]; the variable pass picks by its own x (a variable on +-1 is a boundary literal in every constraint it
// occurs in).  Interior literals get their own scratch rows, as in the other materialising classes.
constexpr int LONG_CLASSES = 7;        // 0..3: one warp per entry, rows 1 / 3 / 5 / 9; 4..6: one LANE per entry (k_long_lane)
__host__ __device__ constexpr int long_lane_cap(int cls) { return cls == 4 ? 8 : cls == 5 ? 16 : 32; }   // interior literals
__host__ __device__ constexpr int long_class_rows(int cls) { return cls == 0 ? 1 : cls == 1 ? 3 : cls == 2 ? 5 : 9; }
// largest Leff of a class: its rows hold cells 0 .. 128 rows - 1, the padded list may run 6 entries beyond Leff
__host__ __device__ constexpr int long_class_maxleff(int cls) { return 128 * long_class_rows(cls) - 8; }

struct LongLists {
    uint4* items[LONG_CLASSES];   // (constraint, restart, nB0 | nBr << 16, nAr)
    int* count;                   // [2][LONG_CLASSES]: set (t & 1) is filled by iteration t, the other one reset
};

template <typename real>
__global__ void __launch_bounds__(128) k_long_scan(const LongCon* __restrict__ cons, int n_long,
                                                   const uint32_t* __restrict__ lits,
                                                   const uint32_t* __restrict__ Sw, const uint32_t* __restrict__ SATw,
                                                   int ntile, int Bp, real* __restrict__ bnd, int32_t* __restrict__ sat,
                                                   real* __restrict__ fe_out, LongLists wl, int set,
                                                   const RunState* __restrict__ rs, const int32_t* __restrict__ goff,
                                                   uint32_t* __restrict__ MI, uint32_t* __restrict__ MT)
{
    const int lane = threadIdx.x & 31;
    if (blockIdx.x == 0 && threadIdx.x < LONG_CLASSES) wl.count[(set ^ 1) * LONG_CLASSES + threadIdx.x] = 0;
    // Grid-stride over the (constraint, tile) pairs of the tiles that hold active restarts: the count lives on the device
    // (the host cannot size the grid by it), and a grid sized for the whole batch spends a late iteration starting and
    // ending CTAs for idle tiles.
    const int atile = rs != nullptr ? min(ntile, (rs->n_act + 31) >> 5) : ntile;
    const long long total = (long long)n_long * atile;
#pragma unroll 1
    for (long long wid = (long long)blockIdx.x * 4 + (threadIdx.x >> 5); wid < total; wid += (long long)gridDim.x * 4) {
    const int c = (int)(wid / atile), tile = (int)(wid % atile);
    const LongCon lc = cons[c];
    const int L = lc.L;
    const uint32_t* lw = lits + lc.off;
    // per group of 32 literals the two bit matrices (literal true, literal interior) are transposed: lane r then holds
    // restart r's bits over the group's literals; their popcounts are the counts, and the words themselves go to
    // MI / MT[group][b] so that the item kernel finds the interior literals of a restart without touching the
    // variables' words again (one coalesced row per group here instead of two scattered sectors per literal there)
    int tc = 0, nBr = 0, nAr = 0;
    const size_t mrow = (size_t)goff[c] * Bp + (size_t)tile * 32 + lane;
    for (int j0 = 0; j0 < L; j0 += 32) {
        const int j = j0 + lane;
        uint32_t tw = 0u, sw = 0xffffffffu;
        if (j < L) {
            const uint32_t w = lw[j];
            const size_t wi = (size_t)(w & LIT_VAR) * ntile + tile;
            const uint32_t s = Sw[wi];
            tw = (w >> 31) ? ~s : s;
            sw = SATw[wi];
        }
        const uint32_t tT = transpose32(tw, lane);
        tc += __popc(tT);
        uint32_t tI = 0u;
        if (__any_sync(FULL, sw != 0xffffffffu)) {
            tI = transpose32(~sw, lane);
            nBr += __popc(tI & tT); nAr += __popc(tI & ~tT);
            MT[mrow + (size_t)(j0 >> 5) * Bp] = tT;
        }
        MI[mrow + (size_t)(j0 >> 5) * Bp] = tI;
    }
    const int nB0 = tc - nBr;
    // lane <-> restart from here on
    const int b = tile * 32 + lane;
    const int Leff = nBr + nAr;
    if (sat && long_pred(lc.type, L, lc.k, nB0 + nBr)) atomicAdd(&sat[b], 1);
    if (Leff == 0) {
        // removing a false literal leaves the point mass at nB0, removing a true one moves it to nB0 - 1
        const int tA = lc.tA - nB0, tB = lc.tB - nB0;
        const real wA = (real)lc.wA * (real)lc.w, wB = (real)lc.wB * (real)lc.w;   // d_t times the constraint's weight
        real* o = bnd + ((size_t)c * Bp + b) * 2;
        o[0] = (tA == 0 ? wA : real(0)) + (tB == 0 ? wB : real(0));
        o[1] = (tA == -1 ? wA : real(0)) + (tB == -1 ? wB : real(0));
        if (fe_out) fe_out[(size_t)c * Bp + b] = long_pred(lc.type, L, lc.k, nB0) ? -(real)lc.w : (real)lc.w;
    }
    const int cls = Leff == 0 ? -1 : Leff <= long_lane_cap(4) ? 4 : Leff <= long_lane_cap(5) ? 5 : Leff <= long_lane_cap(6) ? 6
                  : Leff <= long_class_maxleff(0) ? 0 : Leff <= long_class_maxleff(1) ? 1
                  : Leff <= long_class_maxleff(2) ? 2 : 3;
    const unsigned lt = (1u << lane) - 1u;
#pragma unroll
    for (int k = 0; k < LONG_CLASSES; ++k) {
        const unsigned m = __ballot_sync(FULL, cls == k);
        if (m) {
            int base = 0;
            if (lane == 0) base = atomicAdd(&wl.count[set * LONG_CLASSES + k], __popc(m));
            base = __shfl_sync(FULL, base, 0);
            if (cls == k) wl.items[k][base + __popc(m & lt)] = make_uint4((unsigned)c, (unsigned)b, (unsigned)nB0 | ((unsigned)nBr << 16), (unsigned)nAr);
        }
    }
    }   // grid-stride loop
}

// WPC warps per CTA, each with its own list / pmf buffers of LS / QS entries; persistent over the class's work list.
template <typename real, int NR, int WPC>
__global__ void __launch_bounds__(WPC * 32) k_long_items(const LongCon* __restrict__ cons,
                                                         const uint32_t* __restrict__ lits, const int32_t* __restrict__ slots,
                                                         const real* __restrict__ XT, const uint32_t* __restrict__ Sw,
                                                         const uint32_t* __restrict__ SATw, int ntile, int Bp,
                                                         real* __restrict__ lrows, int row0, int nl, real* __restrict__ bnd,
                                                         real* __restrict__ fe_out, const uint4* __restrict__ items,
                                                         const int* __restrict__ count, int LS, int QS,
                                                         unsigned long long* __restrict__ work,
                                                         const int32_t* __restrict__ goff, const uint32_t* __restrict__ MI,
                                                         const uint32_t* __restrict__ MT)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    real* RcAll = reinterpret_cast<real*>(smem_raw);              // [WPC][LS]  ratios in list order, then gradients
    real* AAll = RcAll + WPC * LS;                                // [WPC][QS]  the pmf
    uint16_t* JAll = reinterpret_cast<uint16_t*>(AAll + WPC * QS);   // [WPC][LS]  literal index at each list position
    constexpr unsigned FULLM = 0xffffffffu;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    real* Rc = RcAll + warp * LS;
    real* Aw = AAll + warp * QS;
    uint16_t* J = JAll + warp * LS;
    const unsigned lt = (1u << lane) - 1u;
    const int n_items = *count;
#pragma unroll 1
    for (int it = blockIdx.x * WPC + warp; it < n_items; it += gridDim.x * WPC) {
        const uint4 ent = items[it];
        const int c = (int)ent.x, b = (int)ent.y;
        const int nB0 = (int)(ent.z & 0xffffu), nBr = (int)(ent.z >> 16), nAr = (int)ent.w;
        const LongCon lc = cons[c];
        const int L = lc.L;
        const uint32_t* lw = lits + lc.off;
        const int32_t* sw = slots + lc.off;
        const int Leff = nBr + nAr;
        // lists [B interior, pad | A interior, pad] of literal indices, from the restart's masks the scan kernel wrote:
        // lane <-> group of 32 literals, positions by a warp scan of the popcounts, every lane expands its own bits.
        // x is gathered for the listed literals only.
        const int nBr4 = (nBr + 3) & ~3, nAr4 = (nAr + 3) & ~3, send = nBr4 + nAr4;
        {
            int pBr = 0, pAr = nBr4;
            const int ngr = (L + 31) >> 5;
            const size_t mrow = (size_t)goff[c] * Bp + b;
            for (int g0 = 0; g0 < ngr; g0 += 32) {
                const int g = g0 + lane;
                uint32_t mi = 0u, mt = 0u;
                if (g < ngr) {
                    mi = MI[mrow + (size_t)g * Bp];
                    if (mi) mt = MT[mrow + (size_t)g * Bp];
                }
                uint32_t mB = mi & mt, mA = mi & ~mt;
                const int cB = __popc(mB), cA = __popc(mA);
                int sB = cB, sA = cA;   // inclusive scans
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int uB = __shfl_up_sync(FULLM, sB, o), uA = __shfl_up_sync(FULLM, sA, o);
                    if (lane >= o) { sB += uB; sA += uA; }
                }
                int qB = pBr + sB - cB, qA = pAr + sA - cA;
                while (mB) { J[qB++] = (uint16_t)(g * 32 + __ffs(mB) - 1); mB &= mB - 1; }
                while (mA) { J[qA++] = (uint16_t)(g * 32 + __ffs(mA) - 1); mA &= mA - 1; }
                pBr += __shfl_sync(FULLM, sB, 31); pAr += __shfl_sync(FULLM, sA, 31);
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
                const bool tb = e < nBr4;
                R = (tb ? u : p) * recip(tb ? p : u);
            }
            Rc[e] = R;
        }
        // ---- S2: forward pmf of the interior literals
        const int off = (3 - Leff) & 3;
        {
            real fe;
            if (NR == 1 && Leff <= 63) fe = long_forward_small<real, 2>(lc, L, Rc, Aw, nBr, nBr4, nAr, Leff, nB0, off, lane, QS, fe_out != nullptr);
            else if (NR == 1) fe = long_forward_small<real, 4>(lc, L, Rc, Aw, nBr, nBr4, nAr, Leff, nB0, off, lane, QS, fe_out != nullptr);
            else fe = long_forward<real, NR>(lc, L, Rc, Aw, nBr, nBr4, send, Leff, nB0, off, lane, QS, fe_out != nullptr);
            if (fe_out) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) fe += __shfl_xor_sync(FULLM, fe, o);
                if (lane == 0) fe_out[(size_t)c * Bp + b] = fe * (real)lc.w;
            }
        }
        __syncwarp();
        // ---- S3 + S5: leave-one-out
        const bool useA = lc.wA != 0.f, useB = lc.wB != 0.f;
        // capture points in true-count index space, t1 <= t2 (equal if only one is used)
        int t1 = lc.tA, t2 = lc.tB;
        real w1 = (real)lc.wA * (real)lc.w, w2 = (real)lc.wB * (real)lc.w;   // d_t times the constraint's weight
        if (!useA) { t1 = t2; w1 = real(0); }
        if (!useB) { t2 = t1; w2 = w1; w1 = real(0); }
        if (t1 > t2) { int tt = t1; t1 = t2; t2 = tt; real ww = w1; w1 = w2; w2 = ww; }
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
        __syncwarp();
        // ---- S5 + write-out of the interior literals' rows
        for (int e = lane; e < send; e += 32) {
            const int j = J[e];
            if (j != 0xffff) {
                const real g = Rc[e];
                // rows of the LONG class are tile-major, [tile][row][32]: the rows of one variable are consecutive, so the
                // variable-side pass (k_glong) streams them instead of touching one 128-byte piece per 8 KB
                lrows[((size_t)(b >> 5) * nl + (size_t)(sw[j] - row0)) * 32 + (b & 31)] = (lw[j] >> 31) ? -g : g;
            }
        }
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------------------------
// k_long_lane: work-list entries with few interior literals (classes 4, 5), one LANE per entry -- any 32 entries of the
// list share a warp, each lane with its own constraint, restart and lists (lane-private columns of shared memory).  The
// loops run to the warp's maximum with per-lane predicates; which entries share a warp enters no result.
//   pmf     q_t <- q_t u + q_{t-1} p over the entry's interior literals in literal order (u = (1+y)/2, p = (1-y)/2),
//   chains  leave-one-out in the stable direction, divisor max(u, p) >= 1/2 (as cm_body_small),
// boundary literals are exact shifts: one pair per (constraint, restart).  Columns: [0, cap] pmf | cap y | cap g | cap j.
// ---------------------------------------------------------------------------------------------------------------------
template <typename real>
__global__ void __launch_bounds__(256) k_long_lane(const LongCon* __restrict__ cons, const uint32_t* __restrict__ lits,
                                                   const int32_t* __restrict__ slots, const real* __restrict__ XT, int Bp,
                                                   real* __restrict__ lrows, int row0, int nl, real* __restrict__ bnd,
                                                   real* __restrict__ fe_out, const uint4* __restrict__ items,
                                                   const int* __restrict__ count, int cap,
                                                   const int32_t* __restrict__ goff, const uint32_t* __restrict__ MI,
                                                   const uint32_t* __restrict__ MT, unsigned long long* __restrict__ work)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpc = blockDim.x >> 5;
    const real half = real(0.5), one = real(1), zero = real(0);
    const size_t per_warp = (size_t)(3 * cap + 1) * 32 * sizeof(real) + (size_t)cap * 32 * sizeof(uint16_t);
    real* q = reinterpret_cast<real*>(smem_raw + warp * per_warp) + lane;    // q[t * 32]
    real* yl = q + (cap + 1) * 32;
    real* gl = yl + cap * 32;
    uint16_t* jl = reinterpret_cast<uint16_t*>(gl - lane + cap * 32) + lane;
    const int n_items = *count;
#pragma unroll 1
    for (int it0 = (blockIdx.x * wpc + warp) * 32; it0 < n_items; it0 += gridDim.x * wpc * 32) {
        const bool have = it0 + lane < n_items;
        const uint4 ent = have ? items[it0 + lane] : make_uint4(0u, 0u, 0u, 0u);
        const int c = (int)ent.x, b = (int)ent.y;
        const int nB0 = (int)(ent.z & 0xffffu), nI = have ? (int)(ent.z >> 16) + (int)ent.w : 0;
        const LongCon lc = cons[c];
        const int L = have ? lc.L : 0;
        const uint32_t* lw = lits + lc.off;
        const int32_t* sw = slots + lc.off;
        // ---- interior literal indices, in literal order, from the entry's masks
        {
            const int ngr = (L + 31) >> 5, ngr_max = __reduce_max_sync(FULL, ngr);
            const size_t mrow = (size_t)goff[c] * Bp + b;
            int pos = 0;
            for (int g = 0; g < ngr_max; ++g) {
                uint32_t mi = g < ngr ? MI[mrow + (size_t)g * Bp] : 0u;
                while (__any_sync(FULL, mi != 0u)) {
                    if (mi) { jl[pos * 32] = (uint16_t)(g * 32 + __ffs(mi) - 1); ++pos; mi &= mi - 1; }
                }
            }
        }
        const int maxI = __reduce_max_sync(FULL, nI);
        // ---- their values (two dependent loads each, independent across the loop)
#pragma unroll 4
        for (int e = 0; e < maxI; ++e) {
            if (e < nI) {
                const uint32_t w = lw[jl[e * 32]];
                const real x = XT[(size_t)(w & LIT_VAR) * Bp + b];
                yl[e * 32] = (w >> 31) ? -x : x;
            }
        }
        // ---- forward pmf; lanes with fewer literals append neutral factors (u = 1, p = 0: exact)
        q[0] = one;
        for (int t = 1; t <= maxI; ++t) q[t * 32] = zero;
        for (int e = 0; e < maxI; ++e) {
            const real y = e < nI ? yl[e * 32] : one;
            const real u = fma(half, y, half), p = fma(-half, y, half);
            real hi = zero;
            for (int t = e + 1; t >= 1; --t) {
                const real lo = q[(t - 1) * 32];
                q[t * 32] = fma(lo, p, hi * u);
                hi = lo;
            }
            q[0] = hi * u;
        }
        if (fe_out && have) {
            real f = zero;
            for (int t = 0; t <= nI; ++t) {
                const real v = q[t * 32];
                f += long_pred(lc.type, L, lc.k, t + nB0) ? -v : v;   // sp = -1 where satisfied
            }
            fe_out[(size_t)c * Bp + b] = f * (real)lc.w;
        }
        const real wA = (real)lc.wA * (real)lc.w, wB = (real)lc.wB * (real)lc.w;   // zero where the target is unused
        const int cA = lc.tA - nB0, cB = lc.tB - nB0;    // targets inside the reduced pmf
        if (work) {   // timing mode: the counted algorithmic work, 6 Leff Keff per entry (as k_long_items)
            unsigned long long fl = 0ull;
            const int keff = lc.k - nB0;
            if (have && (lc.wA != 0.f || lc.wB != 0.f) && keff >= (lc.type == AFS_EK ? 0 : 1) && keff <= nI) {
                int K = min(keff, nI - keff + 1) + 1;
                fl = 6ull * (unsigned long long)nI * (unsigned long long)(K < 1 ? 1 : K);
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) fl += __shfl_xor_sync(FULL, fl, o);
            if (lane == 0 && fl) atomicAdd(work + (blockIdx.x & 31u), fl);
        }
        if (have) {   // boundary literals: removing a false one leaves q, removing a true one takes one shift away
            auto qat = [&](int tau) -> real { return (tau >= 0 && tau <= nI) ? q[tau * 32] : zero; };
            real* o = bnd + ((size_t)c * Bp + b) * 2;
            o[0] = wA * qat(cA) + wB * qat(cB);
            o[1] = wA * qat(cA + 1) + wB * qat(cB + 1);
        }
        // ---- interior literals: one chain each, in the stable direction; two literals per round (independent chains)
        {
            // steps a chain needs: up to the later of the two capture points (top-down chains count from nI - 1)
            const int hiT = max(wA != zero ? cA : -1, wB != zero ? cB : -1), loT = min(wA != zero ? cA : nI, wB != zero ? cB : nI);
            for (int e0 = 0; e0 < maxI; e0 += 2) {
                bool has[2], fwd[2];
                real rb[2], R[2], acc[2], vA[2], vB[2];
                int need = 0;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    has[h] = e0 + h < nI;
                    const real y = has[h] ? yl[(e0 + h) * 32] : one;
                    const real u = fma(half, y, half), p = fma(-half, y, half);
                    fwd[h] = !(y < zero);
                    rb[h] = recip(fwd[h] ? u : p);
                    R[h] = -((fwd[h] ? p : u) * rb[h]);
                    acc[h] = zero; vA[h] = zero; vB[h] = zero;
                    const int nd = has[h] ? (fwd[h] ? min(hiT, nI - 1) + 1 : min(nI - 1 - loT, nI - 1) + 1) : 0;
                    need = max(need, nd);
                }
                const int steps_w = __reduce_max_sync(FULL, need);
                for (int s = 0; s < steps_w; ++s) {
                    const bool in = s <= nI - 1;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const bool on = has[h] && in;
                        const int row = fwd[h] ? s : nI - s;
                        const real a = on ? q[row * 32] : zero;
                        acc[h] = fma(R[h], acc[h], a);
                        const int idx = fwd[h] ? s : nI - 1 - s;        // index of q^(-j) this step completes
                        vA[h] = (on && idx == cA) ? acc[h] : vA[h];
                        vB[h] = (on && idx == cB) ? acc[h] : vB[h];
                    }
                }
#pragma unroll
                for (int h = 0; h < 2; ++h)
                    if (has[h]) gl[(e0 + h) * 32] = (wA * vA[h] + wB * vB[h]) * rb[h];
            }
        }
        // ---- S5 + write-out of the interior literals' rows (tile-major rows of the class)
        for (int e = 0; e < maxI; ++e) {
            if (e < nI) {
                const int j = jl[e * 32];
                const real g = gl[e * 32];
                lrows[((size_t)(b >> 5) * nl + (size_t)(sw[j] - row0)) * 32 + (b & 31)] = (lw[j] >> 31) ? -g : g;
            }
        }
        __syncwarp();
    }
}

}  // namespace afs
