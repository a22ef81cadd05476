// afs_gm.cuh -- per-constraint gradient magnitudes ("adaptive constraint weighting -- informed by
// per-constraint gradient magnitudes"; L188 (i); reading G25):
//     gm[k] = sum_b sum_j | dFE_k/dy_j (X_b) |      (unweighted, l1 over the literals, summed over the batch)
// After the push kernels of an evaluation have run with unit weights, every class reduces its own constraints to one
// partial per (constraint, restart tile) -- lane <-> restart, xor-butterfly sum: a fixed order -- and k_gm_final adds
// the tiles of a constraint in order.  No float atomics.
#pragma once
#include "afs_bits.cuh"
#include "afs_internal.h"

namespace afs {

template <typename real>
__device__ __forceinline__ real warp_sum(real v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
}

// MED / CMED: the literals' gradients sit in their scratch rows.  REC = MedCon or LongCon (off, L).
template <typename real, typename REC>
__global__ void __launch_bounds__(128) k_gm_rows(const REC* __restrict__ cons, int nc, const int32_t* __restrict__ slots,
                                                 const int32_t* __restrict__ ids, const real* __restrict__ scratch, int Bp,
                                                 int B, real* __restrict__ part)
{
    const int lane = threadIdx.x & 31, tile = blockIdx.y, ntile = Bp >> 5;
    const int c = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (c >= nc) return;
    const REC rc = cons[c];
    const int b = tile * 32 + lane;
    real s = real(0);
    for (int j = 0; j < rc.L; ++j) s += fabs(scratch[(size_t)slots[rc.off + j] * Bp + b]);
    s = warp_sum<real>(b < B ? s : real(0));
    if (lane == 0) part[(size_t)ids[c] * ntile + tile] = s;
}

// PULL: nothing is materialised; the leave-one-out products of a clause of at most 5 literals are formed directly.
template <typename real>
__global__ void __launch_bounds__(128) k_gm_pull(const PullClause* __restrict__ cons, int nc, const int32_t* __restrict__ ids,
                                                 const real* __restrict__ XT, int Bp, int B, real* __restrict__ part)
{
    const int lane = threadIdx.x & 31, tile = blockIdx.y, ntile = Bp >> 5;
    const int c = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (c >= nc) return;
    const PullClause pc = cons[c];
    const int L = (int)(pc.hdr & 7u), kind = (int)((pc.hdr >> 3) & 3u);
    const int b = tile * 32 + lane;
    real y[PULL_MAX_LEN];
#pragma unroll
    for (int j = 0; j < PULL_MAX_LEN; ++j) {
        y[j] = real(1);
        if (j < L) {
            const real x = XT[(size_t)(pc.lit[j] & LIT_VAR) * Bp + b];
            y[j] = (pc.lit[j] >> 31) ? -x : x;
        }
    }
    real s = real(0);
#pragma unroll
    for (int j = 0; j < PULL_MAX_LEN; ++j) {
        if (j < L) {
            real pu = real(1), pp = real(1), py = real(1);
#pragma unroll
            for (int i = 0; i < PULL_MAX_LEN; ++i)
                if (i < L && i != j) {
                    pu *= real(0.5) + real(0.5) * y[i]; pp *= real(0.5) - real(0.5) * y[i]; py *= y[i];
                }
            s += fabs(kind == (int)PH_KIND_OR ? pu : kind == (int)PH_KIND_XOR ? py : pu - pp);
        }
    }
    s = warp_sum<real>(b < B ? s : real(0));
    if (lane == 0) part[(size_t)ids[c] * ntile + tile] = s;
}

// LONG: warp = (constraint, tile).  Boundary literals share the pair bnd[c][b]; their numbers per restart come from the
// words as in k_long_scan; interior literals have their own (tile-major) rows.
template <typename real>
__global__ void __launch_bounds__(128) k_gm_long(const LongCon* __restrict__ cons, int n_long,
                                                 const uint32_t* __restrict__ lits, const int32_t* __restrict__ slots,
                                                 const int32_t* __restrict__ ids, const uint32_t* __restrict__ Sw,
                                                 const uint32_t* __restrict__ SATw, int ntile, int Bp, int B,
                                                 const real* __restrict__ lrows, int row0, int nl,
                                                 const real* __restrict__ bnd, real* __restrict__ part)
{
    const int lane = threadIdx.x & 31;
    const long long wid = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
    if (wid >= (long long)n_long * ntile) return;
    const int c = (int)(wid / ntile), tile = (int)(wid % ntile);
    const LongCon lc = cons[c];
    const int L = lc.L, b = tile * 32 + lane;
    int nBt = 0, nI = 0;
    real s = real(0);
    for (int j0 = 0; j0 < L; j0 += 32) {
        const int j = j0 + lane;
        uint32_t tw = 0u, sw = 0xffffffffu;
        if (j < L) {
            const uint32_t w = lits[lc.off + j];
            const size_t wi = (size_t)(w & LIT_VAR) * ntile + tile;
            const uint32_t sg = Sw[wi];
            tw = (w >> 31) ? ~sg : sg;
            sw = SATw[wi];
        }
        const uint32_t tT = transpose32(tw, lane);
        uint32_t tI = transpose32(~sw, lane);           // this restart's interior literals of the group
        nBt += __popc(tT & ~tI); nI += __popc(tI);
        while (__any_sync(FULL, tI != 0u)) {
            if (tI) {
                const int jj = j0 + __ffs(tI) - 1;
                s += fabs(lrows[((size_t)tile * nl + (size_t)(slots[lc.off + jj] - row0)) * 32 + lane]);
                tI &= tI - 1;
            }
        }
    }
    const real* pr = bnd + ((size_t)c * Bp + b) * 2;
    s += fabs(pr[0]) * (real)(L - nBt - nI) + fabs(pr[1]) * (real)nBt;
    s = warp_sum<real>(b < B ? s : real(0));
    if (lane == 0) part[(size_t)ids[c] * ntile + tile] = s;
}

template <typename real>
__global__ void k_gm_final(const real* __restrict__ part, int m, int ntile, real* __restrict__ gm)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
    double acc = 0.0;
    for (int t = 0; t < ntile; ++t) acc += (double)part[(size_t)k * ntile + t];
    gm[k] = (real)acc;
}

}  // namespace afs
