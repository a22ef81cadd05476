// afs_kernels.cuh -- the streaming-path kernels (one launch per phase per step), templated on the arithmetic type
// (float = product, double = fp64 verification build).  Working layout: XT[n][Bp], restart fastest, so that lane <->
// restart gives one 128-byte line per (variable, 32 restarts) -- the "coalesced restart-major gathers" of
// BASELINE.json.  P:Lnn = PAPER.md line nn.
#pragma once
#include "afs_internal.h"
#include "afs_bits.cuh"
#include "afs_retire.cuh"

namespace afs {

constexpr int VAR_WARPS = 4;   // warps per CTA in the variable pass (8 CTAs per SM; measured 2-3 % ahead of 8 warps x 4 CTAs)
constexpr int VAR_VPW = 4;     // consecutive variables per warp

// Is the constraint true when t of its L literals are true?  (Table 2; XOR parity k, G2)
__device__ __forceinline__ bool pred(int type, int L, int k, int t)
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

template <typename real>
__device__ __forceinline__ real ldx(const real* __restrict__ XT, uint32_t w, int Bp, int b)
{
    return XT[(size_t)(w & LIT_VAR) * Bp + b];
}

// ------------------------------------------------------------------------------------------------------------------
// layout changes at the API boundary: X[B,n] <-> XT[n][Bp]
// ------------------------------------------------------------------------------------------------------------------
// Also writes the sign / saturation words of the iterate (Sw, SATw: [n][Bp/32], may be NULL).
template <typename real>
__global__ void __launch_bounds__(256) k_transpose_in(const real* __restrict__ X, real* __restrict__ XT, int B, int n,
                                                      int Bp, const int8_t* __restrict__ mask,
                                                      uint32_t* __restrict__ Sw, uint32_t* __restrict__ SATw,
                                                      int mask_stride = 0, int8_t* __restrict__ maskT = nullptr)
{   // mask_stride = 0: one mask[n] for all restarts; = n: masks[B][n], one per restart (then also written transposed
    // to maskT[n][Bp] for the variable pass)
    __shared__ real tile[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int v0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
    // columns behind the batch (ragged last tile) are copies of the last restart: whatever a warp decides for its 32
    // restarts together (e.g. which body to run) is then a function of the caller's X alone, and a resumed run repeats it
    for (int r = ty; r < 32; r += 8) {
        int b = min(b0 + r, B - 1), v = v0 + tx;
        real x = real(0);
        if (v < n) x = X[(size_t)b * n + v] + real(0);   // + 0 turns -0.0 into +0.0 (G13)
        tile[r][tx] = x;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        int v = v0 + r, b = b0 + tx;
        if (v < n) {
            real x = tile[tx][r];
            if (mask) {   // fixed at entry
                int mk = mask[(size_t)min(b, B - 1) * mask_stride + v];
                mk = mk > 0 ? 1 : mk < 0 ? -1 : 0;   // any positive value means fixed False (+1), any negative fixed True
                if (mk != 0) x = (real)mk;
                if (maskT) maskT[(size_t)v * Bp + b] = (int8_t)mk;
            }
            XT[(size_t)v * Bp + b] = x;
        }
        if (Sw) {   // the 32 lanes of a warp hold one variable's tile (v is warp-uniform)
            const real xx = v < n ? tile[tx][r] : real(0);
            real xm = xx;
            if (mask && v < n) {
                int mk = mask[(size_t)min(b, B - 1) * mask_stride + v];
                mk = mk > 0 ? 1 : mk < 0 ? -1 : 0;
                if (mk != 0) xm = (real)mk;
            }
            const unsigned sb = __ballot_sync(FULL, xm < real(0)), sa = __ballot_sync(FULL, xm == real(1) || xm == real(-1));
            if (tx == 0 && v < n) { Sw[(size_t)v * (Bp >> 5) + blockIdx.y] = sb; SATw[(size_t)v * (Bp >> 5) + blockIdx.y] = sa; }
        }
    }
}

template <typename real>
__global__ void __launch_bounds__(256) k_transpose_out(const real* __restrict__ XT, real* __restrict__ X, int B, int n,
                                                       int Bp)
{
    __shared__ real tile[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int v0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
    for (int r = ty; r < 32; r += 8) {
        int v = v0 + r;
        tile[r][tx] = v < n ? XT[(size_t)v * Bp + b0 + tx] : real(0);
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        int b = b0 + r, v = v0 + tx;
        if (b < B && v < n) X[(size_t)b * n + v] = tile[tx][r];
    }
}

// rounded assignment int8[B,n] from XT (S9): x < 0 -> -1 (True), else +1
template <typename real>
__global__ void __launch_bounds__(256) k_assign_out(const real* __restrict__ XT, int8_t* __restrict__ assign, int B,
                                                    int n, int Bp)
{
    __shared__ int8_t tile[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int v0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
    for (int r = ty; r < 32; r += 8) {
        int v = v0 + r;
        real x = v < n ? XT[(size_t)v * Bp + b0 + tx] : real(0);
        tile[r][tx] = x < real(0) ? -1 : 1;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        int b = b0 + r, v = v0 + tx;
        if (b < B && v < n) assign[(size_t)b * n + v] = tile[tx][r];
    }
}

// ------------------------------------------------------------------------------------------------------------------
// S9 alone: satisfied-constraint count of one iterate, every constraint through the generic forward CSR.
// Integer arithmetic only; thread = (constraint, restart), lanes over restarts.
// ------------------------------------------------------------------------------------------------------------------
template <typename real>
__global__ void __launch_bounds__(256) k_count(const CountCon* __restrict__ cons, const uint32_t* __restrict__ lits,
                                               int m, const real* __restrict__ XT, int Bp, int32_t* __restrict__ sat,
                                               const RunState* __restrict__ rs)
{
    __shared__ int s_sat[8][32];
    if (tile_idle(rs, blockIdx.y)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y * 32 + lane;
    int cnt = 0;
    for (int c = blockIdx.x * 8 + warp; c < m; c += gridDim.x * 8) {
        CountCon cc = cons[c];
        int t = 0;
        for (int j = 0; j < cc.L; ++j) {
            uint32_t w = lits[cc.off + j];
            real x = ldx(XT, w, Bp, b);
            t += ((x < real(0)) != ((w >> 31) != 0)) ? 1 : 0;
        }
        cnt += pred(cc.type, cc.L, cc.k, t) ? 1 : 0;
    }
    s_sat[warp][lane] = cnt;
    __syncthreads();
    if (warp == 0) {
        int tot = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) tot += s_sat[w][lane];
        if (tot) atomicAdd(&sat[b], tot);
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Accessors: the constraint bodies below are written once and read x / write gradients through these, so the
// streaming kernels (global XT[n][Bp], global scratch) and the tile-resident kernel (shared memory) share them.
// ------------------------------------------------------------------------------------------------------------------
template <typename real>
struct XGlobal {
    const real* __restrict__ p;
    int stride, col;
    __device__ __forceinline__ real operator()(uint32_t var) const { return p[(size_t)var * stride + col]; }
};
template <typename real>
struct SGlobal {
    real* __restrict__ p;
    int stride, col;
    __device__ __forceinline__ void put(int slot, real v) const { p[(size_t)slot * stride + col] = v; }
    __device__ __forceinline__ real get(int slot) const { return p[(size_t)slot * stride + col]; }
};

// ------------------------------------------------------------------------------------------------------------------
// CMED class: EK / CARD with L <= CM_MAX_LEN, thread = (constraint, restart).  The pmf q_0..q_L of the number of true
// literals (count basis, G10) lives in the warp's shared-memory buffer, cell t of this lane at q[t * 32]
// (column = lane: conflict-free, and the index may be dynamic, so nothing is padded and nothing is unrolled).
//   forward   q_t <- q_t u_j + q_{t-1} p_j for every literal, one LDS + FMUL + FFMA + STS per cell.
//   gradient  dFE/dy_j = wA q^(-j)_{tA} + wB q^(-j)_{tB} (at most two non-zero d_t).  q^(-j) comes from q by
//             removing literal j in the STABLE direction: s_t = q_t - (p/u) s_{t-1} from the bottom when p <= 1/2
//             (q^(-j)_t = s_t / u), z_i = q_{L-i} - (u/p) z_{i-1} from the top otherwise (q^(-j)_{L-1-i} = z_i / p).
//             Every lane walks its own direction through its own column in ONE loop (the ratio is <= 1 and the
//             divisor >= 1/2 either way: nothing that vanishes at x = +-1 is divided by); the loop ends at the later
//             of the two directions' capture points, which depend on the constraint only (warp-uniform).
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float rcp_rn(float x) { return __frcp_rn(x); }
__device__ __forceinline__ double rcp_rn(double x) { return 1.0 / x; }

template <typename real, typename XL, typename SW>
__device__ __forceinline__ void cm_body(const LongCon& lc, const uint32_t* __restrict__ lw,
                                        const int32_t* __restrict__ sw, const XL& xl, const SW& sc,
                                        real* __restrict__ q, int& satcnt, real& fe, const bool want_fe,
                                        const bool commit = true)
{
    // commit = false: this lane's restart was served by cm_body_small; it walks along (the loops are warp-uniform)
    // but writes no result
    const real half = real(0.5), one = real(1), zero = real(0);
    const int L = lc.L;
    q[0] = one;
    int tc = 0;
    for (int j = 0; j < L; ++j) {
        const uint32_t w = lw[j];
        const real x = xl(w & LIT_VAR);
        const bool neg = (w >> 31) != 0;
        tc += ((x < zero) != neg) ? 1 : 0;
        const real y = neg ? -x : x;
        const real u = fma(half, y, half), p = fma(-half, y, half);
        // cells j+1 .. 1, four at a time with the loads in front (the stores of a group never feed its loads)
        real hi = zero;   // old q_{t}, starting with q_{j+1} = 0
        int t = j + 1;
        for (; t >= 4; t -= 4) {
            const real l1 = q[(t - 1) * 32], l2 = q[(t - 2) * 32], l3 = q[(t - 3) * 32], l4 = q[(t - 4) * 32];
            q[t * 32] = fma(l1, p, mul_rn(hi, u));
            q[(t - 1) * 32] = fma(l2, p, mul_rn(l1, u));
            q[(t - 2) * 32] = fma(l3, p, mul_rn(l2, u));
            q[(t - 3) * 32] = fma(l4, p, mul_rn(l3, u));
            hi = l4;
        }
        for (; t >= 1; --t) {
            const real lo = q[(t - 1) * 32];
            q[t * 32] = fma(lo, p, mul_rn(hi, u));
            hi = lo;
        }
        q[0] = mul_rn(hi, u);
    }
    satcnt += (commit && pred(lc.type, L, lc.k, tc)) ? 1 : 0;
    if (want_fe) {
        real f = zero;
        for (int t = 0; t <= L; ++t) {
            const real v = q[t * 32];
            f += (lc.type == AFS_CARD ? t >= lc.k : t == lc.k) ? -v : v;   // sp_t = -1 where satisfied
        }
        if (commit) fe = mul_rn(f, (real)lc.w);
    } else if (commit) {
        fe = zero;
    }
    const bool useA = lc.wA != 0.f, useB = lc.wB != 0.f;
    if (!useA && !useB) {   // constant expansion (CARD k = 0 or k = L+1, G5): zero gradient
        for (int j = 0; j < L; ++j)
            if (commit) sc.put(sw[j], zero);
        return;
    }
    const int tA = useA ? lc.tA : lc.tB, tB = useB ? lc.tB : lc.tA;   // tA <= tB
    const real wA = useA ? (real)lc.wA : zero, wB = useB ? (real)lc.wB : zero;
    // capture steps: bottom-up chain step = t; top-down chain step i <-> t = L-1-i
    const int f1 = tA, f2 = tB, b1 = L - 1 - tB, b2 = L - 1 - tA;
    const int bp0 = min(f1, b1), bp3 = max(f2, b2);
    const int m1 = max(f1, b1), m2 = min(f2, b2);
    const int bp[4] = {bp0, min(m1, m2), max(m1, m2), bp3};
    // two literals at a time: two independent chains per lane, loads of a group of four steps in front
    for (int j0 = 0; j0 < L; j0 += 2) {
        real R[2], rb[2], w1[2], w2[2], acc[2], v1[2], v2[2];
        const real* qp[2];
        int st[2], c1[2], c2[2];
        bool ng[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int j = min(j0 + h, L - 1);
            const uint32_t w = lw[j];
            const real x = xl(w & LIT_VAR);
            ng[h] = (w >> 31) != 0;
            const real y = ng[h] ? -x : x;
            const real u = fma(half, y, half), p = fma(-half, y, half);
            const bool fwd = !(y < zero);   // p <= 1/2
            rb[h] = rcp_rn(fwd ? u : p);
            R[h] = -mul_rn(fwd ? p : u, rb[h]);
            c1[h] = fwd ? f1 : b1; c2[h] = fwd ? f2 : b2;
            w1[h] = fwd ? wA : wB; w2[h] = fwd ? wB : wA;
            qp[h] = fwd ? q : q + L * 32;
            st[h] = fwd ? 32 : -32;
            acc[h] = zero; v1[h] = zero; v2[h] = zero;
        }
        int s = 0;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int e = bp[b];
            if (e >= s) {
                int cnt = e - s + 1;
                for (; cnt >= 4; cnt -= 4) {
                    real a[2][4];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
#pragma unroll
                        for (int i = 0; i < 4; ++i) a[h][i] = qp[h][i * st[h]];
                        qp[h] += 4 * st[h];
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        acc[0] = fma(R[0], acc[0], a[0][i]);
                        acc[1] = fma(R[1], acc[1], a[1][i]);
                    }
                }
                for (; cnt > 0; --cnt) {
                    const real a0 = *qp[0], a1 = *qp[1];
                    qp[0] += st[0]; qp[1] += st[1];
                    acc[0] = fma(R[0], acc[0], a0);
                    acc[1] = fma(R[1], acc[1], a1);
                }
                s = e + 1;
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    v1[h] = c1[h] == e ? acc[h] : v1[h];
                    v2[h] = c2[h] == e ? acc[h] : v2[h];
                }
            }
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (j0 + h < L) {
                const real g = mul_rn(mul_rn(fma(w1[h], v1[h], mul_rn(w2[h], v2[h])), rb[h]), (real)lc.w);
                if (commit) sc.put(sw[j0 + h], ng[h] ? -g : g);
            }
        }
    }
}

// The same constraint when few of its literals are strictly inside the cube -- the usual state of a PGD iterate after a
// few dozen steps (clipping): a literal on the boundary is the factor 1 (y = +1) or z (y = -1) of
// Q(z) = prod (u_j + p_j z), an exact shift, so only the interior literals (at most `cap` per restart, lane-private
// lists in the same shared-memory buffer) go through the pmf and the chains; all boundary literals of a kind share one
// gradient value.  The decision is per restart (lane), so that a restart's result never depends on which restarts share
// its warp: returns the mask of lanes served here; lanes with more interior literals than the buffer holds write
// nothing and are served by cm_body (commit = their complement).
// Buffer rows: [0, cap] pmf | [cap+1, 2cap] y | [2cap+1, 3cap] gradients.
template <typename real, typename XL, typename SW>
__device__ __forceinline__ unsigned cm_body_small(const LongCon& lc, const uint32_t* __restrict__ lw,
                                              const int32_t* __restrict__ sw, const XL& xl, const SW& sc,
                                              real* __restrict__ q, const int qrows, int& satcnt, real& fe,
                                              const bool want_fe)
{
    const real half = real(0.5), one = real(1), zero = real(0);
    const int L = lc.L;
    const int cap = min(12, (qrows - 1) / 3);
    if (cap < 1) return 0u;
    real* __restrict__ yl = q + (cap + 1) * 32;
    real* __restrict__ gl = yl + cap * 32;
    int nB0 = 0, nI = 0, tc = 0;
    for (int j = 0; j < L; ++j) {
        const uint32_t w = lw[j];
        const real x = xl(w & LIT_VAR);
        const bool neg = (w >> 31) != 0;
        tc += ((x < zero) != neg) ? 1 : 0;
        const real y = neg ? -x : x;
        if (y == -one) ++nB0;
        else if (y != one) { if (nI < cap) yl[nI * 32] = y; ++nI; }
    }
    const bool mine = nI <= cap;
    const unsigned served = __ballot_sync(FULL, mine);
    if (served == 0u) return 0u;
    const int maxI = __reduce_max_sync(FULL, mine ? nI : 0);
    satcnt += (mine && pred(lc.type, L, lc.k, tc)) ? 1 : 0;
    // forward pmf of the interior literals; lanes with fewer of them append neutral factors (u = 1, p = 0: exact)
    q[0] = one;
    for (int t = 1; t <= maxI; ++t) q[t * 32] = zero;
    for (int e = 0; e < maxI; ++e) {
        const real y = (mine && e < nI) ? yl[e * 32] : one;
        const real u = fma(half, y, half), p = fma(-half, y, half);
        real hi = zero;
        for (int t = e + 1; t >= 1; --t) {
            const real lo = q[(t - 1) * 32];
            q[t * 32] = fma(lo, p, mul_rn(hi, u));
            hi = lo;
        }
        q[0] = mul_rn(hi, u);
    }
    if (want_fe) {
        real f = zero;
        for (int t = 0; t <= maxI; ++t) {
            const real v = q[t * 32];
            f += (lc.type == AFS_CARD ? t + nB0 >= lc.k : t + nB0 == lc.k) ? -v : v;   // sp = -1 where satisfied
        }
        if (mine) fe = mul_rn(f, (real)lc.w);
    } else if (mine) {
        fe = zero;
    }
    const real wA = (real)lc.wA, wB = (real)lc.wB;   // zero where the target is unused
    const int cA = lc.tA - nB0, cB = lc.tB - nB0;    // targets inside the reduced pmf (true-count index minus the shift)
    // boundary literals: removing a false one leaves q, removing a true one takes one shift away
    real gA0, gB0;
    {
        const real a0 = (cA >= 0 && cA <= maxI) ? q[cA * 32] : zero, a1 = (cA + 1 >= 0 && cA + 1 <= maxI) ? q[(cA + 1) * 32] : zero;
        const real b0 = (cB >= 0 && cB <= maxI) ? q[cB * 32] : zero, b1 = (cB + 1 >= 0 && cB + 1 <= maxI) ? q[(cB + 1) * 32] : zero;
        gA0 = fma(wA, a0, mul_rn(wB, b0));
        gB0 = fma(wA, a1, mul_rn(wB, b1));
    }
    // interior literals: leave-one-out in the stable direction (divisor max(u, p) >= 1/2), one chain per literal
    for (int e = 0; e < maxI; ++e) {
        const bool has = e < nI && mine;
        const real y = has ? yl[e * 32] : one;
        const real u = fma(half, y, half), p = fma(-half, y, half);
        const bool fwd = !(y < zero);
        const real rb = rcp_rn(fwd ? u : p);
        const real R = -mul_rn(fwd ? p : u, rb);
        real acc = zero, vA = zero, vB = zero;
        for (int s = 0; s < maxI; ++s) {
            const bool on = has && s <= nI - 1;
            const int row = fwd ? s : nI - s;
            const real a = on ? q[row * 32] : zero;
            acc = fma(R, acc, a);
            const int idx = fwd ? s : nI - 1 - s;        // index of q^(-j) this step completes
            vA = (on && idx == cA) ? acc : vA;
            vB = (on && idx == cB) ? acc : vB;
        }
        if (has) gl[e * 32] = mul_rn(fma(wA, vA, mul_rn(wB, vB)), rb);
    }
    // S5 + write-out in literal order
    int e = 0;
    for (int j = 0; j < L; ++j) {
        const uint32_t w = lw[j];
        const real x = xl(w & LIT_VAR);
        const bool neg = (w >> 31) != 0;
        const real y = neg ? -x : x;
        real g;
        if (y == one) g = gA0;
        else if (y == -one) g = gB0;
        else { g = gl[min(e, cap - 1) * 32]; ++e; }
        g = mul_rn(g, (real)lc.w);
        if (mine) sc.put(sw[j], neg ? -g : g);
    }
    return served;
}

// ------------------------------------------------------------------------------------------------------------------
// MED class: OR / XOR beyond the pull lengths and NAE / EO / AMO of any length; thread = (constraint, restart).
// Division-free leave-one-out by prefix x suffix (BASELINE.json subsystem (2)): a forward pass over the literals
// writes the prefix state in front of literal j to a private row (aux0 / aux1, one row per literal of the class), a
// backward pass carries the suffix state in registers, combines and writes dFE/dy_j (times the literal sign, S5) to
// the literal's scratch row.  State: OR / XOR the running product (u = (1+y)/2 resp. y); NAE the products of u and
// of p = (1-y)/2; EO / AMO the pmf of the true count truncated to {0, 1} (count basis, G10; d_t of P:L52):
//   OR   FE = 2 prod u - 1                 dFE/dy_j = prod_{i!=j} u_i
//   XOR  FE = s prod y                     dFE/dy_j = s prod_{i!=j} y_i                    (s = +1 odd parity, -1 even)
//   NAE  FE = 2 prod u + 2 prod p - 1      dFE/dy_j = prod_{i!=j} u_i - prod_{i!=j} p_i
//   EO   FE = 1 - 2 q_1                    dFE/dy_j = q_0^(-j) - q_1^(-j)
//   AMO  FE = 1 - 2 (q_0 + q_1)            dFE/dy_j = - q_1^(-j)
// Two short dynamic loops, no register arrays: any length, a few hundred bytes of code.
// ------------------------------------------------------------------------------------------------------------------
template <typename real, typename XL, typename SW>
__device__ __forceinline__ void med_body(const MedCon& mc, const uint32_t* __restrict__ lc,
                                         const int32_t* __restrict__ sc, const XL& xl, const SW& sw, const SW& ax0,
                                         const SW& ax1, int& satcnt, real& fe)
{
    const real half = real(0.5), one = real(1), zero = real(0);
    const int L = mc.L, row0 = mc.off;
    const int type = mc.type;
    const real wk = (real)mc.w;   // eq. (5) weight; 1 unless the problem was created with weights (x * 1 is exact)
    int t = 0;
    if (type == AFS_OR || type == AFS_XOR) {
        const bool is_or = type == AFS_OR;
        const real s = is_or ? one : ((mc.k & 1) ? one : -one);
        real pre = one;
#pragma unroll 2
        for (int j = 0; j < L; ++j) {
            const uint32_t w = lc[j];
            const real x = xl(w & LIT_VAR);
            const bool neg = (w >> 31) != 0;
            t += ((x < zero) != neg) ? 1 : 0;
            const real y = neg ? -x : x;
            ax0.put(row0 + j, pre);
            pre = mul_rn(pre, is_or ? fma(half, y, half) : y);
        }
        fe = is_or ? fma(real(2), pre, -one) : mul_rn(s, pre);
        real suf = s;
#pragma unroll 2
        for (int j = L - 1; j >= 0; --j) {
            const uint32_t w = lc[j];
            const real x = xl(w & LIT_VAR);
            const bool neg = (w >> 31) != 0;
            const real y = neg ? -x : x;
            const real g = mul_rn(ax0.get(row0 + j), suf);
            sw.put(sc[j], mul_rn(neg ? -g : g, wk));
            suf = mul_rn(suf, is_or ? fma(half, y, half) : y);
        }
    } else if (type == AFS_NAE) {
        real pu = one, pp = one;
#pragma unroll 2
        for (int j = 0; j < L; ++j) {
            const uint32_t w = lc[j];
            const real x = xl(w & LIT_VAR);
            const bool neg = (w >> 31) != 0;
            t += ((x < zero) != neg) ? 1 : 0;
            const real y = neg ? -x : x;
            ax0.put(row0 + j, pu);
            ax1.put(row0 + j, pp);
            pu = mul_rn(pu, fma(half, y, half));
            pp = mul_rn(pp, fma(-half, y, half));
        }
        fe = fma(real(2), pu, fma(real(2), pp, -one));
        real su = one, sp = one;
#pragma unroll 2
        for (int j = L - 1; j >= 0; --j) {
            const uint32_t w = lc[j];
            const real x = xl(w & LIT_VAR);
            const bool neg = (w >> 31) != 0;
            const real y = neg ? -x : x;
            const real g = fma(ax0.get(row0 + j), su, -mul_rn(ax1.get(row0 + j), sp));
            sw.put(sc[j], mul_rn(neg ? -g : g, wk));
            su = mul_rn(su, fma(half, y, half));
            sp = mul_rn(sp, fma(-half, y, half));
        }
    } else {   // EO, AMO
        const bool is_eo = type == AFS_EO;
        real a0 = one, a1 = zero;
#pragma unroll 2
        for (int j = 0; j < L; ++j) {
            const uint32_t w = lc[j];
            const real x = xl(w & LIT_VAR);
            const bool neg = (w >> 31) != 0;
            t += ((x < zero) != neg) ? 1 : 0;
            const real y = neg ? -x : x;
            const real u = fma(half, y, half), p = fma(-half, y, half);
            ax0.put(row0 + j, a0);
            ax1.put(row0 + j, a1);
            a1 = fma(a1, u, mul_rn(a0, p));
            a0 = mul_rn(a0, u);
        }
        fe = is_eo ? fma(real(-2), a1, one) : fma(real(-2), a0 + a1, one);
        real s0 = one, s1 = zero;
#pragma unroll 2
        for (int j = L - 1; j >= 0; --j) {
            const uint32_t w = lc[j];
            const real x = xl(w & LIT_VAR);
            const bool neg = (w >> 31) != 0;
            const real y = neg ? -x : x;
            const real u = fma(half, y, half), p = fma(-half, y, half);
            const real P0 = ax0.get(row0 + j), P1 = ax1.get(row0 + j);
            const real q0 = mul_rn(P0, s0);
            const real q1 = fma(P1, s0, mul_rn(P0, s1));
            const real g = is_eo ? q0 - q1 : -q1;
            sw.put(sc[j], mul_rn(neg ? -g : g, wk));
            s1 = fma(s1, u, mul_rn(s0, p));
            s0 = mul_rn(s0, u);
        }
    }
    satcnt += pred(type, L, mc.k, t) ? 1 : 0;
    fe = mul_rn(fe, wk);
}

template <typename real>
__global__ void __launch_bounds__(128) k_med(const MedCon* __restrict__ cons, int c_begin, int c_end,
                                             const uint32_t* __restrict__ lits, const int32_t* __restrict__ slots,
                                             const real* __restrict__ XT, int Bp, real* __restrict__ scratch,
                                             real* __restrict__ aux0, real* __restrict__ aux1,
                                             int32_t* __restrict__ sat, real* __restrict__ fe_out,
                                             const RunState* __restrict__ rs)
{
    __shared__ int s_sat[4][32];
    if (tile_idle(rs, blockIdx.y)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y * 32 + lane;
    int satcnt = 0;
    const XGlobal<real> xl{XT, Bp, b};
    const SGlobal<real> sc{scratch, Bp, b}, a0{aux0, Bp, b}, a1{aux1, Bp, b};
    for (int c = c_begin + blockIdx.x * 4 + warp; c < c_end; c += gridDim.x * 4) {
        const MedCon mc = cons[c];
        real fe;
        med_body<real>(mc, lits + mc.off, slots + mc.off, xl, sc, a0, a1, satcnt, fe);
        if (fe_out) fe_out[(size_t)c * Bp + b] = fe;
    }
    if (sat) {
        s_sat[warp][lane] = satcnt;
        __syncthreads();
        if (warp == 0) {
            int tot = s_sat[0][lane] + s_sat[1][lane] + s_sat[2][lane] + s_sat[3][lane];
            if (tot) atomicAdd(&sat[b], tot);
        }
    }
}

template <typename real>
__global__ void __launch_bounds__(128) k_cmed(const LongCon* __restrict__ cons, int c_begin, int c_end,
                                              const uint32_t* __restrict__ lits, const int32_t* __restrict__ slots,
                                              const real* __restrict__ XT, int Bp, real* __restrict__ scratch,
                                              int32_t* __restrict__ sat, real* __restrict__ fe_out, int qrows,
                                              const RunState* __restrict__ rs)
{
    extern __shared__ __align__(16) unsigned char cm_smem[];
    __shared__ int s_sat[4][32];
    if (tile_idle(rs, blockIdx.y)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y * 32 + lane;
    int satcnt = 0;
    const XGlobal<real> xl{XT, Bp, b};
    const SGlobal<real> sc{scratch, Bp, b};
    real* q = reinterpret_cast<real*>(cm_smem) + (size_t)warp * qrows * 32 + lane;
    for (int c = c_begin + blockIdx.x * 4 + warp; c < c_end; c += gridDim.x * 4) {
        const LongCon lc = cons[c];
        real fe;
        const unsigned served = cm_body_small<real>(lc, lits + lc.off, slots + lc.off, xl, sc, q, qrows, satcnt, fe, fe_out != nullptr);
        if (served != FULL)
            cm_body<real>(lc, lits + lc.off, slots + lc.off, xl, sc, q, satcnt, fe, fe_out != nullptr, !((served >> lane) & 1u));
        if (fe_out) fe_out[(size_t)c * Bp + b] = fe;
    }
    if (sat) {
        s_sat[warp][lane] = satcnt;
        __syncthreads();
        if (warp == 0) {
            int tot = s_sat[0][lane] + s_sat[1][lane] + s_sat[2][lane] + s_sat[3][lane];
            if (tot) atomicAdd(&sat[b], tot);
        }
    }
}

// ------------------------------------------------------------------------------------------------------------------
// Variable pass: thread = (variable, restart), lanes over 32 restarts of one variable.  Fuses
//   S1-S3,S5 for the PULL class: the leave-one-out product of every occurrence is recomputed from the other
//        literals (no scratch, no atomics); occurrences come in runs of equal shape so the inner loops are
//        branch-free; the warp stages 32 entries with one coalesced load and gathers several occurrences at once,
//   S6   deterministic segmented reduction of the materialised gradients over the transposed CSR (fixed order),
//   S7-S8 step, clip, fixed-variable mask,
//   S9   sign bits of X_t (one ballot word per variable and restart tile; the counts of the PULL clauses are taken
//        from these words by k_sat_pull),
//   S10  merge of the previous iterate into the best-so-far (its count is complete once the previous launches ended).
// EVAL = true is afs_eval_grad: writes G^T instead of stepping.
// ------------------------------------------------------------------------------------------------------------------
template <typename real>
struct VarArgs {
    int n, Bp, t;
    const int32_t* pull_ptr;
    const uint32_t* pull_words;
    const int32_t* run_ptr;
    const uint32_t* runs;
    const float* gconst;
    const int32_t* slot_ptr;
    const real* scratch;
    const real* Xin;
    real* Xout;
    real lr;
    const int8_t* mask;
    const int32_t* sat_prev;     // counts of X_{t-1}, or NULL when there is nothing to merge
    int32_t* sat_zero;           // the count row of X_{t+1} (ring of three), zeroed here; may be NULL
    const int32_t* best_sat_in;
    int32_t* best_sat_out;
    const int32_t* best_step_in;
    int32_t* best_step_out;
    const uint32_t* S_prev;      // sign words of X_{t-1} (best-so-far merge)
    uint32_t* S_next;            // sign / saturation words of X_{t+1}, written with the step (may alias S_prev: the same
    uint32_t* SAT_next;          // thread reads a word of S_prev before it writes that word of S_next)
    uint32_t* best_bits;
    const real* GL;              // LONGT: [n][Bp] the LONG class's share of the gradient (k_glong)
    const int8_t* maskT;         // CONV variant only: per-restart masks [n][Bp] (afs_pgd_run_masks), or NULL
    // CONV (afs_pgd_run_conv): a restart stops after the first step with max_v |dX| < tol (G24)
    real tol;
    const int32_t* conv_in;      // [Bp] number of steps after which the restart stopped, -1 = still running
    int32_t* conv_out;
    const void* delta_prev;      // [Bp] DBits: max |dX| of the previous step, NULL = already folded into conv_in
    void* delta_cur;             // [Bp] DBits: max |dX| of this step (integer atomicMax), zeroed by the previous pass
    void* delta_zero;            // [Bp] the row of the next step
    const RunState* rs;          // tile groups behind the active restarts return at once (afs_retire.cuh); may be NULL
    int32_t* moved;              // non-NULL on the iterations a retirement follows: moved[b] = 1 if any x_v changed
    real* GT;
};

// |dX| as an order-preserving unsigned integer (non-negative IEEE values compare like their bit patterns), so that the
// per-restart maximum over all variables is an integer atomicMax: exact and independent of the order of arrival
__device__ __forceinline__ unsigned int dbits(float d) { return __float_as_uint(d); }
__device__ __forceinline__ unsigned long long dbits(double d) { return (unsigned long long)__double_as_longlong(d); }
template <typename real> struct DBits;
template <> struct DBits<float> { typedef unsigned int type; static __device__ __forceinline__ float val(unsigned int u) { return __uint_as_float(u); } };
template <> struct DBits<double> { typedef unsigned long long type; static __device__ __forceinline__ double val(unsigned long long u) { return __longlong_as_double((long long)u); } };

template <typename real> struct Pair;
template <> struct Pair<float> { typedef float2 type; };
template <> struct Pair<double> { typedef double2 type; };

__device__ __forceinline__ float flip(float x, uint32_t signbit) { return __int_as_float(__float_as_int(x) ^ (int)signbit); }
__device__ __forceinline__ double flip(double x, uint32_t signbit) { return signbit ? -x : x; }

// Per-entry auxiliary word, decoded once per staged chunk (one entry per lane):
//   fp32 OR/NAE: the bits of h = +-0.5 (sign = literal negated), so that u = h x + 0.5;   fp32 XOR: the sign mask
//   fp64 (verification build): just the negation flag
template <typename real, int KIND>
__device__ __forceinline__ uint32_t pull_aux(uint32_t w)
{
    if (sizeof(real) == 4 && KIND != (int)PH_KIND_XOR) return 0x3f000000u | (w & PE_NEG);
    return w & PE_NEG;
}
__device__ __forceinline__ float pull_u(float x, uint32_t aux) { return fmaf(__int_as_float((int)aux), x, 0.5f); }
__device__ __forceinline__ double pull_u(double x, uint32_t aux) { return (aux ? -0.5 : 0.5) * x + 0.5; }
__device__ __forceinline__ float pull_p(float x, uint32_t aux) { return fmaf(-__int_as_float((int)aux), x, 0.5f); }
__device__ __forceinline__ double pull_p(double x, uint32_t aux) { return 0.5 - (aux ? -0.5 : 0.5) * x; }

constexpr int PULL_SBUF = 48;   // uint2 slots per warp: 32 staged entries + slack for the unrolled tail (kept valid)

// One run: `count` occurrences of NOTHER other literals each, entries at words[beg ...).  xcol points at column b of
// the X matrix (global XT or a shared-memory tile), rowbytes is its row pitch in bytes (rows * rowbytes < 2^32).
// The warp loads 32 entries with one coalesced load, every lane decodes its entry (byte offset of the row, sign
// material) into the warp's shared staging buffer, and all lanes then walk the occurrences reading whole records
// with one broadcast LDS each.  Returns the run's contribution to dF/dx_v (carrying the own literal's sign).
// Column loaders: byte offset of a row -> x of this lane's restart.  Global: column b of XT[n][Bp]; shared: column
// `lane` of the tile X[n][32] of the resident kernel (32-bit shared-window address, LDS).
template <typename real>
struct ColGlobal {
    const char* __restrict__ base;
    // c = sub-tile of 32 restarts handled by the same lane (RPL > 1): 32 elements further along the row
    __device__ __forceinline__ real at(uint32_t off, int c = 0) const
    {
        return *reinterpret_cast<const real*>(base + off + c * 32 * (int)sizeof(real));
    }
};
template <typename real>
struct ColShared {
    uint32_t base;
    __device__ __forceinline__ real at(uint32_t off, int = 0) const
    {
        real v;
        if constexpr (sizeof(real) == 4) asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(base + off));
        else asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(base + off));
        return v;
    }
};

// RPL = restart sub-tiles per lane: the lane works on restarts lane, lane + 32, ... of a tile of 32 * RPL restarts,
// so every staged entry, every offset and every branch is paid once for RPL gathers.  g[c] += the run's contribution.
template <typename real, int KIND, int NOTHER, int RPL, typename COL>
__device__ __forceinline__ void pull_run(const uint32_t* __restrict__ words, int beg, int count, const COL& xcol,
                                         uint32_t rowbytes, int lane, uint2* sbuf, real (&gout)[RPL])
{
    constexpr int OPC = 32 / NOTHER;              // occurrences per staged chunk of <= 32 entries
    // occurrences gathered together: 8 (NOTHER <= 2) or up to 16 loads in flight per lane.  Wider batches were measured
    // slower at the same register count (configs[3]: 272 -> 320 us per iteration with twice the batch): their tails
    // gather rows that are discarded, and occupancy already hides the latency (see k_var)
    constexpr int U0 = NOTHER <= 2 ? 4 : 2;
    // one sub-tile per lane (the resident kernel): four occurrences per batch whatever their length -- fewer, longer
    // loop bodies (configs[1]: 80.6 -> 67.3 us per iteration against 2 for the 3- and 4-literal runs; 8/5/4: 69.9)
    constexpr int U = RPL == 1 ? 4 : (U0 / RPL >= 1 ? U0 / RPL : 1);
    real g[RPL];
#pragma unroll
    for (int c = 0; c < RPL; ++c) g[c] = real(0);
    for (int o0 = 0; o0 < count; o0 += OPC) {
        const int nocc = min(OPC, count - o0);
        const uint32_t wm = words[beg + o0 * NOTHER + lane];   // reading past the run is harmless (valid entries / padding)
        // the sign flag rides in bit 0 of the first offset of an occurrence; entries past the chunk (staged only so
        // that the unrolled tail reads valid rows) must not carry it, or the tail's loads would be misaligned
        const uint32_t sgn = lane < nocc * NOTHER ? (wm >> 30) & 1u : 0u;
        sbuf[lane] = make_uint2((wm & PE_VAR) * rowbytes | sgn, pull_aux<real, KIND>(wm));
        __syncwarp();
        for (int o = 0; o < nocc; o += U) {
            uint2 e[U][NOTHER];
            real x[U][NOTHER][RPL];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const uint2* rec = sbuf + (o + u) * NOTHER;
                if (NOTHER == 2) {
                    uint4 t = *reinterpret_cast<const uint4*>(rec);
                    e[u][0] = make_uint2(t.x, t.y); e[u][NOTHER - 1] = make_uint2(t.z, t.w);
                } else if (NOTHER == 4) {
                    uint4 t0 = *reinterpret_cast<const uint4*>(rec), t1 = *reinterpret_cast<const uint4*>(rec + 2);
                    e[u][0] = make_uint2(t0.x, t0.y); e[u][1 % NOTHER] = make_uint2(t0.z, t0.w);
                    e[u][2 % NOTHER] = make_uint2(t1.x, t1.y); e[u][3 % NOTHER] = make_uint2(t1.z, t1.w);
                } else {
#pragma unroll
                    for (int i = 0; i < NOTHER; ++i) e[u][i] = rec[i];
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u)
#pragma unroll
                for (int i = 0; i < NOTHER; ++i) {
                    const uint32_t off = i == 0 ? (e[u][0].x & ~1u) : e[u][i].x;
#pragma unroll
                    for (int c = 0; c < RPL; ++c) x[u][i][c] = xcol.at(off, c);
                }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const bool live = o + u < nocc;
#pragma unroll
                for (int c = 0; c < RPL; ++c) {
                    real d;
                    if (KIND == (int)PH_KIND_XOR) {
                        real prod = flip(x[u][0][c], e[u][0].y);
#pragma unroll
                        for (int i = 1; i < NOTHER; ++i) prod *= flip(x[u][i][c], e[u][i].y);
                        d = prod;
                    } else {
                        real pu = pull_u(x[u][0][c], e[u][0].y);
#pragma unroll
                        for (int i = 1; i < NOTHER; ++i) pu *= pull_u(x[u][i][c], e[u][i].y);
                        d = pu;
                        if (KIND == (int)PH_KIND_NAE) {
                            real pp = pull_p(x[u][0][c], e[u][0].y);
#pragma unroll
                            for (int i = 1; i < NOTHER; ++i) pp *= pull_p(x[u][i][c], e[u][i].y);
                            d = pu - pp;
                        }
                    }
                    d = flip(d, e[u][0].x << 31);
                    if (live) g[c] += d;
                }
            }
        }
        __syncwarp();
    }
#pragma unroll
    for (int c = 0; c < RPL; ++c) gout[c] += g[c];
}

// all runs of one variable: g[c] += sum over the runs (each run summed on its own first, in stream order)
template <typename real, int RPL, typename COL>
__device__ __forceinline__ void pull_variable(const uint32_t* __restrict__ runs, int rbeg, int rend,
                                              const uint32_t* __restrict__ words, int wbeg, const COL& xcol,
                                              uint32_t rowbytes, int lane, uint2* sbuf, real (&g)[RPL])
{
    real acc[RPL];
#pragma unroll
    for (int c = 0; c < RPL; ++c) acc[c] = real(0);
    int pos = wbeg;
    for (int r = rbeg; r < rend; ++r) {
        const uint32_t d = runs[r];
        const int count = (int)(d & 0x07ffffffu), nother = (int)((d >> 27) & 7u), kind = (int)(d >> 30);
#define AFS_RUN(K, N) pull_run<real, K, N, RPL, COL>(words, pos, count, xcol, rowbytes, lane, sbuf, acc)
        if (kind == (int)PH_KIND_OR) {
            switch (nother) { case 1: AFS_RUN(0, 1); break; case 2: AFS_RUN(0, 2); break; case 3: AFS_RUN(0, 3); break; default: AFS_RUN(0, 4); break; }
        } else if (kind == (int)PH_KIND_XOR) {
            switch (nother) { case 1: AFS_RUN(1, 1); break; case 2: AFS_RUN(1, 2); break; case 3: AFS_RUN(1, 3); break; default: AFS_RUN(1, 4); break; }
        } else {
            switch (nother) { case 1: AFS_RUN(2, 1); break; case 2: AFS_RUN(2, 2); break; case 3: AFS_RUN(2, 3); break; default: AFS_RUN(2, 4); break; }
        }
#undef AFS_RUN
        pos += count * nother;
    }
#pragma unroll
    for (int c = 0; c < RPL; ++c) g[c] += acc[c];
}

// 32 warps per SM at <= 64 registers: the pass waits on L2 gathers, and occupancy is what hides them -- at
// 95 registers (2 CTAs per SM) the same code took 1.5x as long on configs[3] (measured: 420 -> 274 us per iteration).
// LONGT: the instance has LONG-class constraints; their share of the gradient comes summed from k_glong.
template <typename real, bool EVAL, int RPL, bool LONGT, bool CONV>
__global__ void __launch_bounds__(VAR_WARPS * 32, 32 / VAR_WARPS) k_var(const VarArgs<real> a)
{
    __shared__ __align__(16) uint2 s_stage[VAR_WARPS][PULL_SBUF];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tile0 = blockIdx.y * RPL, ntile = a.Bp >> 5;     // this lane's restarts: (tile0 + c) * 32 + lane
    const int b = tile0 * 32 + lane;
    const int Bp = a.Bp;
    const real one = real(1);
    const real* __restrict__ xcol = a.Xin + b;
    const ColGlobal<real> xg{reinterpret_cast<const char*>(xcol)};
    if (tile_idle(a.rs, tile0)) return;       // first thing: late in a run most CTAs of the grid are of this kind
    uint2* sbuf = s_stage[warp];
    for (int i = lane; i < PULL_SBUF; i += 32) sbuf[i] = make_uint2(0u, 0u);   // slack slots must stay valid offsets
    __syncwarp();
    const int vbeg = (blockIdx.x * VAR_WARPS + warp) * VAR_VPW;
    const int vend = min(vbeg + VAR_VPW, a.n);
    // ---- convergence detection: a restart whose last step stayed below tol is frozen from now on
    typedef typename DBits<real>::type dbits_t;
    bool frozen[RPL];
    real dmax[RPL];
#pragma unroll
    for (int c = 0; c < RPL; ++c) {
        frozen[c] = false; dmax[c] = real(0);
        if (CONV) {
            frozen[c] = a.conv_in[b + 32 * c] >= 0;
            if (!frozen[c] && a.delta_prev)
                frozen[c] = DBits<real>::val(static_cast<const dbits_t*>(a.delta_prev)[b + 32 * c]) < a.tol;
        }
    }
    // ---- S10: did the previous iterate improve on the best so far?
    bool imp[RPL];
    unsigned impmask[RPL];
    int sprev[RPL];
    bool anyimp = false;
#pragma unroll
    for (int c = 0; c < RPL; ++c) {
        imp[c] = false; impmask[c] = 0u; sprev[c] = 0;
        if (!EVAL && a.sat_prev != nullptr) {
            sprev[c] = a.sat_prev[b + 32 * c];
            imp[c] = sprev[c] > a.best_sat_in[b + 32 * c];
            impmask[c] = __ballot_sync(FULL, imp[c]);
            anyimp |= impmask[c] != 0u;
        }
    }
    for (int v = vbeg; v < vend; ++v) {
        if (!EVAL) {
            if (anyimp && lane == 0) {
#pragma unroll
                for (int c = 0; c < RPL; ++c)
                    if (impmask[c]) {
                        size_t wi = (size_t)v * ntile + tile0 + c;
                        a.best_bits[wi] = (a.best_bits[wi] & ~impmask[c]) | (a.S_prev[wi] & impmask[c]);
                    }
            }
            if (v == 0) {
#pragma unroll
                for (int c = 0; c < RPL; ++c) {
                    if (a.sat_zero) a.sat_zero[b + 32 * c] = 0;
                    if (CONV) {   // the step count at which the restart stopped: the previous step was number t
                        const int ci = a.conv_in[b + 32 * c];
                        a.conv_out[b + 32 * c] = ci >= 0 ? ci : (frozen[c] ? a.t : -1);
                        static_cast<dbits_t*>(a.delta_zero)[b + 32 * c] = 0;
                    }
                    int bs = a.best_sat_in[b + 32 * c], stp = a.best_step_in[b + 32 * c];
                    a.best_sat_out[b + 32 * c] = imp[c] ? sprev[c] : bs;
                    a.best_step_out[b + 32 * c] = imp[c] ? a.t - 1 : stp;
                }
            }
        }
        real x[RPL], g[RPL];
        int mk = 0;
#pragma unroll
        for (int c = 0; c < RPL; ++c) x[c] = xcol[(size_t)v * Bp + 32 * c];
        if (!EVAL) mk = a.mask ? a.mask[v] : 0;
        int mkl[RPL];   // per restart (CONV variant with per-restart masks), else the shared value
#pragma unroll
        for (int c = 0; c < RPL; ++c) mkl[c] = (CONV && a.maskT) ? (int)a.maskT[(size_t)v * Bp + b + 32 * c] : mk;
        if (CONV && a.maskT) mk = 0;   // some restart may be free: the gradient is needed
#pragma unroll
        for (int c = 0; c < RPL; ++c) g[c] = real(0);
        if (mk == 0) {   // a fixed variable never moves: its gradient is not needed
            const real gc = (real)a.gconst[v];
#pragma unroll
            for (int c = 0; c < RPL; ++c) g[c] = gc;
            pull_variable<real, RPL>(a.runs, a.run_ptr[v], a.run_ptr[v + 1], a.pull_words, a.pull_ptr[v], xg,
                                     (uint32_t)Bp * (uint32_t)sizeof(real), lane, sbuf, g);
            // ---- S6: materialised gradients of v, fixed (transposed-CSR) order
            const int s1 = a.slot_ptr[v + 1];
            int s = a.slot_ptr[v];
            const real* __restrict__ sc = a.scratch + b;
            for (; s + 4 <= s1; s += 4) {
#pragma unroll
                for (int c = 0; c < RPL; ++c) {
                    real g0 = sc[(size_t)s * Bp + 32 * c], g1 = sc[(size_t)(s + 1) * Bp + 32 * c];
                    real g2 = sc[(size_t)(s + 2) * Bp + 32 * c], g3 = sc[(size_t)(s + 3) * Bp + 32 * c];
                    g[c] += g0; g[c] += g1; g[c] += g2; g[c] += g3;
                }
            }
            for (; s < s1; ++s)
#pragma unroll
                for (int c = 0; c < RPL; ++c) g[c] += sc[(size_t)s * Bp + 32 * c];
            if (LONGT) {   // the LONG class's share of dF/dx_v, summed by k_glong in its own fixed order
#pragma unroll
                for (int c = 0; c < RPL; ++c) g[c] += a.GL[(size_t)v * Bp + b + 32 * c];
            }
        }
#pragma unroll
        for (int c = 0; c < RPL; ++c) {
            if (EVAL) {
                a.GT[(size_t)v * Bp + b + 32 * c] = g[c];
            } else {
                // ---- S7-S8
                real xn = x[c] - a.lr * g[c];
                xn = xn > one ? one : xn;
                xn = xn < -one ? -one : xn;
                if (mkl[c] != 0 || (CONV && frozen[c])) xn = x[c];
                a.Xout[(size_t)v * Bp + b + 32 * c] = xn;
                if (a.moved && xn != x[c]) a.moved[b + 32 * c] = 1;
                if (CONV) dmax[c] = fmax(dmax[c], fabs(xn - x[c]));
                const unsigned sb = __ballot_sync(FULL, xn < real(0)), sa = __ballot_sync(FULL, xn == one || xn == -one);
                if (lane == 0) {
                    a.S_next[(size_t)v * ntile + tile0 + c] = sb;
                    a.SAT_next[(size_t)v * ntile + tile0 + c] = sa;
                }
            }
        }
    }
    if (CONV) {
#pragma unroll
        for (int c = 0; c < RPL; ++c)
            if (dmax[c] > real(0)) atomicMax(static_cast<dbits_t*>(a.delta_cur) + b + 32 * c, dbits(dmax[c]));
    }
}

// ------------------------------------------------------------------------------------------------------------------
// S6 for the LONG class: GL[v][b] = sum over the LONG-class literals of v, in transposed-CSR order.  warp = (variable,
// tile), lane <-> restart.  A literal's gradient is its scratch row only where this restart's x_v is strictly inside the
// cube; on the boundary it is one of the pair bnd[c][b] that the long kernels wrote for ALL boundary literals of the
// constraint, picked by the literal's truth value (a variable on +-1 is a boundary literal in every constraint it
// occurs in).  Eight literals per round, their loads issued together: the pass waits on L2 / HBM latency, not on issue.
// ------------------------------------------------------------------------------------------------------------------
// TPW = restart tiles per warp (the lane works on restarts lane, lane + 32 of a group of TPW tiles): one descriptor
// shuffle and one offset computation serve TPW loads.
template <typename real, int TPW>
__global__ void __launch_bounds__(256) k_glong(int n, int ntile, int Bp, const int32_t* __restrict__ lslot_ptr,
                                               const int32_t* __restrict__ lslot_info, const real* __restrict__ Xin,
                                               const real* __restrict__ lrows /* scratch + nslots_a * Bp: [tile][nl][32] */, int nl,
                                               const real* __restrict__ bnd, const int8_t* __restrict__ mask,
                                               real* __restrict__ GL, const RunState* __restrict__ rs)
{
    const int lane = threadIdx.x & 31;
    // Grid-stride over (variable, group of TPW tiles) for the groups that hold active restarts; the active count lives
    // on the device, so the grid is sized for the SMs, not for the batch (idle tiles cost nothing).
    const int ngrp = rs != nullptr ? min(ntile / TPW, (rs->n_act + 32 * TPW - 1) / (32 * TPW)) : ntile / TPW;
    const long long total = (long long)n * ngrp;
#pragma unroll 1
    for (long long wid = (long long)blockIdx.x * 8 + (threadIdx.x >> 5); wid < total; wid += (long long)gridDim.x * 8) {
    const int v = (int)(wid / ngrp), tile0 = (int)(wid % ngrp) * TPW;
    if (mask && mask[v] != 0) continue;   // a fixed variable never moves: its gradient is not needed
    const int s0 = lslot_ptr[v], s1 = lslot_ptr[v + 1];
    // One base pointer and 32-bit element offsets per lane and tile: a restart on the boundary reads the pair table
    // (second element where the literal is true, i.e. (x < 0) != negated), one inside the cube reads the class's rows.
    const real* __restrict__ base[TPW];
    uint32_t sgn[TPW], neg0[TPW];
    bool onb[TPW];
    real g[TPW];
#pragma unroll
    for (int c = 0; c < TPW; ++c) {
        const int b = (tile0 + c) * 32 + lane;
        const real x = Xin[(size_t)v * Bp + b];
        onb[c] = x == real(1) || x == real(-1);
        neg0[c] = x < real(0) ? 1u : 0u;
        base[c] = onb[c] ? bnd + (size_t)b * 2 : lrows + ((size_t)(tile0 + c) * nl + (size_t)s0) * 32 + lane;
        sgn[c] = onb[c] ? 0x80000000u : 0u;      // chain rule sign (S5) for pair entries; the rows carry it already
        g[c] = real(0);
    }
    const uint32_t pair_stride = (uint32_t)Bp * 2u;
    for (int sb0 = s0; sb0 < s1; sb0 += 32) {
        const int myinfo = sb0 + lane < s1 ? lslot_info[sb0 + lane] : 0;   // 32 descriptors with one coalesced load
        const int cnt = min(32, s1 - sb0);
        int k = 0;
        for (; k + 8 <= cnt; k += 8) {   // eight literals per round, their loads issued together
            real t[8][TPW];
            uint32_t ln[8];
#pragma unroll
            for (int h = 0; h < 8; ++h) {
                const uint32_t info = (uint32_t)__shfl_sync(FULL, myinfo, k + h);
                const uint32_t offB = (info >> 1) * pair_stride, offS = (uint32_t)(sb0 - s0 + k + h) * 32u;
                ln[h] = info & 1u;
#pragma unroll
                for (int c = 0; c < TPW; ++c) t[h][c] = base[c][onb[c] ? offB + (ln[h] ^ neg0[c]) : offS];
            }
#pragma unroll
            for (int h = 0; h < 8; ++h)
#pragma unroll
                for (int c = 0; c < TPW; ++c) g[c] += flip(t[h][c], ln[h] ? sgn[c] : 0u);
        }
        for (; k < cnt; ++k) {
            const uint32_t info = (uint32_t)__shfl_sync(FULL, myinfo, k);
            const uint32_t offB = (info >> 1) * pair_stride, offS = (uint32_t)(sb0 - s0 + k) * 32u, l1 = info & 1u;
#pragma unroll
            for (int c = 0; c < TPW; ++c) g[c] += flip(base[c][onb[c] ? offB + (l1 ^ neg0[c]) : offS], l1 ? sgn[c] : 0u);
        }
    }
#pragma unroll
    for (int c = 0; c < TPW; ++c) GL[(size_t)v * Bp + (tile0 + c) * 32 + lane] = g[c];
    }   // grid-stride loop
}

// ------------------------------------------------------------------------------------------------------------------
// S9 for the PULL class, bit-parallel over restarts: the sign words S[v][tile] (bit r = "x_v < 0" for restart
// tile*32 + r) written by the variable pass give the truth of 32 restarts of a clause with a few logic ops.
// thread = (clause, group of TPT restart tiles), lane <-> clause: the literal words are read once, the TPT sign words
// of a literal are one 4*TPT-byte load, and every load of a clause is independent of the others.  The per-restart
// totals come from a butterfly transposition (bit_column_sums: lane r collects restart r).  Integers only.
// ------------------------------------------------------------------------------------------------------------------
template <int TPT>
struct SWords { uint32_t w[TPT]; };
template <int TPT>
__device__ __forceinline__ SWords<TPT> ld_swords(const uint32_t* __restrict__ p)
{
    SWords<TPT> r;
    if constexpr (TPT == 4) { uint4 t = *reinterpret_cast<const uint4*>(p); r.w[0] = t.x; r.w[1] = t.y; r.w[2] = t.z; r.w[3] = t.w; }
    else if constexpr (TPT == 2) { uint2 t = *reinterpret_cast<const uint2*>(p); r.w[0] = t.x; r.w[1] = t.y; }
    else r.w[0] = *p;
    return r;
}

template <int TPT>
__global__ void __launch_bounds__(256) k_sat_pull(const PullClause* __restrict__ cons, int m,
                                                  const uint32_t* __restrict__ S, int ntile,
                                                  int32_t* __restrict__ sat, const RunState* __restrict__ rs)
{
    __shared__ int s_cnt[TPT][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int tile0 = blockIdx.y * TPT;
    if (tile_idle(rs, tile0)) return;
    if (threadIdx.x < TPT * 32) s_cnt[threadIdx.x >> 5][threadIdx.x & 31] = 0;
    __syncthreads();
    int cnt[TPT];
#pragma unroll
    for (int k = 0; k < TPT; ++k) cnt[k] = 0;
    const int stride = gridDim.x * 256;
    for (int c0 = (blockIdx.x * 8 + warp) * 32; c0 < m; c0 += stride) {
        const int c = c0 + lane;
        uint32_t T[TPT];
#pragma unroll
        for (int k = 0; k < TPT; ++k) T[k] = 0u;
        if (c < m) {
            const uint4* rec = reinterpret_cast<const uint4*>(cons + c);
            const uint4 h0 = rec[0], h1 = rec[1];
            const uint32_t lit[PULL_MAX_LEN] = {h0.y, h0.z, h0.w, h1.x, h1.y};
            const int L = (int)(h0.x & 7u), kind = (int)((h0.x >> 3) & 3u);
            uint32_t vor[TPT], vand[TPT], vxor[TPT];
#pragma unroll
            for (int k = 0; k < TPT; ++k) { vor[k] = 0u; vand[k] = 0xffffffffu; vxor[k] = 0u; }
#pragma unroll
            for (int j = 0; j < PULL_MAX_LEN; ++j)
                if (j < L) {
                    const uint32_t flipm = (lit[j] >> 31) ? 0xffffffffu : 0u;
                    const SWords<TPT> sw = ld_swords<TPT>(S + (size_t)(lit[j] & LIT_VAR) * ntile + tile0);
#pragma unroll
                    for (int k = 0; k < TPT; ++k) {
                        const uint32_t tj = sw.w[k] ^ flipm;
                        vor[k] |= tj; vand[k] &= tj; vxor[k] ^= tj;
                    }
                }
            const uint32_t par = ((h0.x >> 5) & 1u) ? 0xffffffffu : 0u;
#pragma unroll
            for (int k = 0; k < TPT; ++k)
                T[k] = kind == (int)PH_KIND_OR ? vor[k] : kind == (int)PH_KIND_XOR ? ~(vxor[k] ^ par) : (vor[k] & ~vand[k]);
        }
#pragma unroll
        for (int k = 0; k < TPT; ++k) cnt[k] += bit_column_sums(T[k], lane);
    }
#pragma unroll
    for (int k = 0; k < TPT; ++k)
        if (cnt[k]) atomicAdd(&s_cnt[k][lane], cnt[k]);
    __syncthreads();
    if (threadIdx.x < TPT * 32) {
        const int k = threadIdx.x >> 5, r = threadIdx.x & 31;
        const int v = s_cnt[k][r];
        if (v) atomicAdd(&sat[(tile0 + k) * 32 + r], v);
    }
}

// objective of the PULL class for afs_eval_grad (S2, S4): thread = (clause, restart), per-warp partial sums in a
// fixed clause order.  OR 2 prod u - 1;  XOR s prod y;  NAE 2 prod u + 2 prod p - 1.
template <typename real>
__global__ void __launch_bounds__(256) k_fe_pull(const CountCon* __restrict__ cons, const uint32_t* __restrict__ lits,
                                                 int m, const real* __restrict__ XT, int Bp, real* __restrict__ Fpart)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int b = blockIdx.y * 32 + lane;
    const int part = blockIdx.x * 8 + warp, nparts = gridDim.x * 8;
    const real half = real(0.5), one = real(1);
    real acc = real(0);
    for (int c = part; c < m; c += nparts) {
        const CountCon cc = cons[c];
        real pu = one, pp = one, py = one;
        for (int j = 0; j < cc.L; ++j) {
            uint32_t w = lits[cc.off + j];
            real x = ldx(XT, w, Bp, b);
            real y = (w >> 31) ? -x : x;
            pu *= half + half * y; pp *= half - half * y; py *= y;
        }
        acc += cc.type == AFS_OR ? real(2) * pu - one
             : cc.type == AFS_XOR ? ((cc.k & 1) ? py : -py)
                                  : real(2) * pu + real(2) * pp - one;
    }
    Fpart[(size_t)part * Bp + b] = acc;
}

// F[b] = sum of the variable-pass partials, then the medium, then the long expansions -- fixed order, fp64 accumulator
template <typename real>
__global__ void k_reduce_F(const real* __restrict__ Fpart, int nparts, const real* __restrict__ fe_med, int n_med,
                           const real* __restrict__ fe_cm, int n_cm, const real* __restrict__ fe_long, int n_long,
                           int Bp, int B, real* __restrict__ F)
{
    int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= B) return;
    double acc = 0.0;
    for (int i = 0; i < nparts; ++i) acc += (double)Fpart[(size_t)i * Bp + b];
    for (int i = 0; i < n_med; ++i) acc += (double)fe_med[(size_t)i * Bp + b];
    for (int i = 0; i < n_cm; ++i) acc += (double)fe_cm[(size_t)i * Bp + b];
    for (int i = 0; i < n_long; ++i) acc += (double)fe_long[(size_t)i * Bp + b];
    F[b] = (real)acc;
}

// ------------------------------------------------------------------------------------------------------------------
// End of afs_pgd_run: fold the last two iterates into the best-so-far, then write everything in the caller's
// layout: X[B,n], best_assign int8[B,n], best_sat[B], best_step[B].
// ------------------------------------------------------------------------------------------------------------------
template <typename real>
struct FinArgs {
    int n, B, Bp, steps;
    const real* XT;               // X_steps
    const int32_t* sat_prev;      // counts of X_{steps-1} (unused when steps == 0)
    const int32_t* sat_fin;       // counts of X_steps
    const int32_t* best_sat_in;   // best over iterates 0..steps-2
    const int32_t* best_step_in;
    const uint32_t* S_prev;       // sign bits of X_{steps-1}
    const uint32_t* best_bits;
    real* X;
    int8_t* best_assign;
    int32_t* best_sat;
    int32_t* best_step;
    real tol;                     // > 0: convergence detection (afs_pgd_run_conv)
    const int32_t* conv_in;       // [Bp] steps after which the column stopped (-1: running), before the last step is folded
    const void* delta_last;       // [Bp] DBits: max |dX| of the last step, NULL = nothing to fold
    int32_t* conv_step;           // caller's array [B] or NULL
    const RunState* rs;           // only the tiles of active restarts are written (the others were written at retirement)
    const int32_t* orig;          // caller's restart index of every column, -1 = none (pads)
};

template <typename real>
__global__ void __launch_bounds__(256) k_finalize(const FinArgs<real> a)
{
    __shared__ real tile[32][33];
    __shared__ unsigned s_bits[32];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int v0 = blockIdx.x * 32, tileb = blockIdx.y, b0 = tileb * 32, ntile = a.Bp >> 5;
    if (tile_idle(a.rs, tileb)) return;
    const int b = b0 + tx;
    int best = a.best_sat_in[b], bstep = a.best_step_in[b];
    bool imp1 = false;
    if (a.sat_prev != nullptr) {
        int sp = a.sat_prev[b];
        imp1 = sp > best;
        if (imp1) { best = sp; bstep = a.steps - 1; }
    }
    const unsigned m1 = __ballot_sync(FULL, imp1);
    const int sf = a.sat_fin[b];
    const bool imp2 = sf > best;
    if (imp2) { best = sf; bstep = a.steps; }
    const unsigned m2 = __ballot_sync(FULL, imp2);
    for (int r = ty; r < 32; r += 8) {
        int v = v0 + r;
        real x = real(0);
        unsigned bits = 0;
        if (v < a.n) {
            x = a.XT[(size_t)v * a.Bp + b];
            size_t wi = (size_t)v * ntile + tileb;
            bits = a.best_bits[wi];
            if (m1) bits = (bits & ~m1) | (a.S_prev[wi] & m1);
        }
        unsigned fb = __ballot_sync(FULL, x < real(0));
        bits = (bits & ~m2) | (fb & m2);
        tile[r][tx] = x;
        if (tx == 0) s_bits[r] = bits;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        const int bb = a.orig[b0 + r], v = v0 + tx;
        if (bb >= 0 && v < a.n) {
            if (a.X) a.X[(size_t)bb * a.n + v] = tile[tx][r];
            if (a.best_assign) a.best_assign[(size_t)bb * a.n + v] = ((s_bits[tx] >> r) & 1u) ? -1 : 1;
        }
    }
    const int ob = a.orig[b];
    if (blockIdx.x == 0 && ty == 0 && ob >= 0) {
        if (a.best_sat) a.best_sat[ob] = best;
        if (a.best_step) a.best_step[ob] = bstep;
        if (a.conv_step) {
            int cs = -1;
            if (a.tol > real(0)) {
                typedef typename DBits<real>::type dbits_t;
                cs = a.conv_in[b];
                if (cs < 0 && a.delta_last && DBits<real>::val(static_cast<const dbits_t*>(a.delta_last)[b]) < a.tol) cs = a.steps;
            }
            a.conv_step[ob] = cs;
        }
    }
}


}  // namespace afs
