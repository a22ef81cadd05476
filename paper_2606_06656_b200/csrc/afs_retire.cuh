// afs_retire.cuh -- retirement of restarts that have reached a fixed point of the PGD map, and compaction of the rest.
//
// One PGD step is a deterministic function of the restart's own iterate (constant step size, no coupling between
// restarts: PAPER.md L164, L182), so a restart with X_{t+1} = X_t bit for bit will never move again: every later iterate
// equals X_t, rounds to the same assignment and satisfies the same constraints, so neither X nor the best record can
// change ("idling converged elements waste compute").  Every few iterations the streaming path
//   1. folds the pending iterate into the best record of every column and splits the columns into frozen and active
//      ones                                                                              (k_retire_plan, one CTA),
//   2. writes the frozen restarts' results -- X, best assignment, best count and step -- to the caller's arrays, which
//      is exactly what the end of the run would have written for them                               (k_retire_out),
//   3. gathers the active columns to the front of a fresh working set: iterate, sign / saturation words, best-so-far
//      bits                                                                                            (k_compact),
// and every per-iteration kernel returns at once for tiles behind the active ones (the count lives on the device: no
// host round trip).  Results are bit-identical to running every restart for every step; only the work is not done.
#pragma once
#include "afs_bits.cuh"
#include "afs_internal.h"

namespace afs {

struct RunState {      // device-resident bookkeeping of one afs_pgd_run call (streaming path)
    int n_act;         // columns [0, n_act) hold active restarts; [n_act, ceil32(n_act)) copies of column 0 (never output)
    int n_ret;         // entries of the retire list of the last plan
    int pad[2];
};

static __global__ void k_run_init(RunState* rs, int B, int Bp, int32_t* orig, int32_t* moved)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) { rs->n_act = B; rs->n_ret = 0; }
    if (i < Bp) { orig[i] = i < B ? i : -1; moved[i] = 0; }
}

// tiles at or behind this one hold no active restart
__device__ __forceinline__ bool tile_idle(const RunState* rs, int tile) { return rs != nullptr && tile * 32 >= rs->n_act; }

// One CTA.  Column p < n_act: merge iterate t (count sat_t[p]) into the best record; frozen = it did not move in step t.
// Active columns keep their order.  Outputs in the NEW layout: orig_out, best_sat_out, best_step_out, src (old column of
// every new one, pads included); in the OLD layout: imp[p] (iterate t improved the best: its sign bits are the best
// bits), ret[] (frozen columns) with their merged record in ret_sat / ret_step.
static __global__ void __launch_bounds__(1024) k_retire_plan(RunState* rs, int t, const int32_t* __restrict__ sat_t,
                                                      const int32_t* __restrict__ best_sat_in,
                                                      const int32_t* __restrict__ best_step_in,
                                                      const int32_t* __restrict__ orig_in, int32_t* __restrict__ moved,
                                                      int32_t* __restrict__ best_sat_out, int32_t* __restrict__ best_step_out,
                                                      int32_t* __restrict__ orig_out, int32_t* __restrict__ src,
                                                      uint8_t* __restrict__ imp, int32_t* __restrict__ ret,
                                                      int32_t* __restrict__ ret_sat, int32_t* __restrict__ ret_step,
                                                      // convergence detection (tol > 0): the step just taken is folded
                                                      // into the stop count of every column
                                                      double tol, int is64, const void* __restrict__ delta_t,
                                                      const int32_t* __restrict__ conv_in, int32_t* __restrict__ conv_out,
                                                      int32_t* __restrict__ ret_conv)
{
    __shared__ int s_warp[2][32];
    __shared__ int s_base[2];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_act = rs->n_act;
    if (tid < 2) s_base[tid] = 0;
    __syncthreads();
    for (int p0 = 0; p0 < n_act; p0 += 1024) {
        const int p = p0 + tid;
        const bool in = p < n_act;
        int bs = 0, bt = 0;
        bool improved = false, frozen = false;
        if (in) {
            bs = best_sat_in[p]; bt = best_step_in[p];
            const int sp = sat_t[p];
            improved = sp > bs;
            if (improved) { bs = sp; bt = t; }
            frozen = moved[p] == 0;
            imp[p] = improved ? 1 : 0;
        }
        int cs = -1;
        if (in && tol > 0.0) {
            cs = conv_in[p];
            if (cs < 0) {
                const double d = is64 ? __longlong_as_double(static_cast<const long long*>(delta_t)[p])
                                      : (double)__uint_as_float(static_cast<const unsigned int*>(delta_t)[p]);
                if (d < tol) cs = t + 1;
            }
        }
        const unsigned mA = __ballot_sync(FULL, in && !frozen), mR = __ballot_sync(FULL, in && frozen);
        if (lane == 0) { s_warp[0][warp] = __popc(mA); s_warp[1][warp] = __popc(mR); }
        __syncthreads();
        int offA = s_base[0], offR = s_base[1];
        for (int w = 0; w < warp; ++w) { offA += s_warp[0][w]; offR += s_warp[1][w]; }
        const unsigned lt = (1u << lane) - 1u;
        if (in && !frozen) {
            const int q = offA + __popc(mA & lt);
            src[q] = p; orig_out[q] = orig_in[p]; best_sat_out[q] = bs; best_step_out[q] = bt;
            if (tol > 0.0) conv_out[q] = cs;
        }
        if (in && frozen) {
            const int q = offR + __popc(mR & lt);
            ret[q] = p; ret_sat[q] = bs; ret_step[q] = bt; ret_conv[q] = cs;
        }
        __syncthreads();
        if (tid == 0) {
            int a = 0, r = 0;
            for (int w = 0; w < 32; ++w) { a += s_warp[0][w]; r += s_warp[1][w]; }
            s_base[0] += a; s_base[1] += r;
        }
        __syncthreads();
    }
    const int na = s_base[0], nr = s_base[1];
    __syncthreads();
    // pads of the last active tile: copies of the first active column (real dynamics, never output)
    const int na32 = (na + 31) & ~31;
    for (int q = na + tid; q < na32; q += 1024) {
        src[q] = src[0]; orig_out[q] = -1; best_sat_out[q] = best_sat_out[0]; best_step_out[q] = best_step_out[0];
        if (tol > 0.0) conv_out[q] = conv_out[0];
    }
    for (int q = tid; q < na32; q += 1024) moved[q] = 0;
    if (tid == 0) { rs->n_act = na; rs->n_ret = nr; }
}

// Results of the frozen restarts, in the caller's layout.  Block = 32 variables x 32 list entries, lanes along v.
template <typename real>
__global__ void __launch_bounds__(256) k_retire_out(const RunState* __restrict__ rs, int n, int Bp,
                                                    const real* __restrict__ XT, const uint32_t* __restrict__ S_t,
                                                    const uint32_t* __restrict__ best_bits, const uint8_t* __restrict__ imp,
                                                    const int32_t* __restrict__ ret, const int32_t* __restrict__ ret_sat,
                                                    const int32_t* __restrict__ ret_step, const int32_t* __restrict__ orig,
                                                    real* __restrict__ X, int8_t* __restrict__ best_assign,
                                                    int32_t* __restrict__ best_sat, int32_t* __restrict__ best_step,
                                                    const int32_t* __restrict__ ret_conv, int32_t* __restrict__ conv_step)
{
    const int n_ret = rs->n_ret;
    if ((int)blockIdx.y * 32 >= n_ret) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int v = blockIdx.x * 32 + lane, ntile = Bp >> 5;
    for (int e = warp; e < 32; e += 8) {
        const int i = blockIdx.y * 32 + e;
        if (i >= n_ret) break;
        const int p = ret[i], o = orig[p];
        if (o < 0) continue;
        if (v < n) {
            const size_t wi = (size_t)v * ntile + (p >> 5);
            const unsigned bit = ((imp[p] ? S_t[wi] : best_bits[wi]) >> (p & 31)) & 1u;
            if (X) X[(size_t)o * n + v] = XT[(size_t)v * Bp + p];
            if (best_assign) best_assign[(size_t)o * n + v] = bit ? -1 : 1;
        }
        if (blockIdx.x == 0 && lane == 0) {
            if (best_sat) best_sat[o] = ret_sat[i];
            if (best_step) best_step[o] = ret_step[i];
            if (conv_step) conv_step[o] = ret_conv[i];
        }
    }
}

// The active columns gathered to the front of a fresh working set.  warp = (variable, new tile), lane <-> new column.
template <typename real>
__global__ void __launch_bounds__(256) k_compact(const RunState* __restrict__ rs, int n, int Bp,
                                                 const int32_t* __restrict__ src, const uint8_t* __restrict__ imp,
                                                 const real* __restrict__ XT_old, const uint32_t* __restrict__ S_t,
                                                 const uint32_t* __restrict__ bits_old, real* __restrict__ XT_new,
                                                 uint32_t* __restrict__ S_new, uint32_t* __restrict__ SAT_new,
                                                 uint32_t* __restrict__ bits_new)
{
    const int tile = blockIdx.y;
    if (tile * 32 >= rs->n_act) return;
    const int lane = threadIdx.x & 31, ntile = Bp >> 5;
    const int v = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (v >= n) return;
    const int s = src[tile * 32 + lane];
    const real x = XT_old[(size_t)v * Bp + s];
    XT_new[(size_t)v * Bp + tile * 32 + lane] = x;
    const size_t wi = (size_t)v * ntile + (s >> 5);
    const unsigned bit = ((imp[s] ? S_t[wi] : bits_old[wi]) >> (s & 31)) & 1u;
    const unsigned sb = __ballot_sync(FULL, x < real(0)), sa = __ballot_sync(FULL, x == real(1) || x == real(-1));
    const unsigned bb = __ballot_sync(FULL, bit != 0u);
    if (lane == 0) {
        const size_t wo = (size_t)v * ntile + tile;
        S_new[wo] = sb; SAT_new[wo] = sa; bits_new[wo] = bb;
    }
}

// Per-restart masks (afs_pgd_run_masks) follow their restarts: the rows of maskT[n][Bp] gathered like the iterate.
// warp = (variable, new tile), lane <-> new column; pads take the mask of the column they copy.
static __global__ void __launch_bounds__(256) k_compact_mask(const RunState* __restrict__ rs, int n, int Bp,
                                                             const int32_t* __restrict__ src,
                                                             const int8_t* __restrict__ mask_old,
                                                             int8_t* __restrict__ mask_new)
{
    const int tile = blockIdx.y;
    if (tile * 32 >= rs->n_act) return;
    const int lane = threadIdx.x & 31;
    const int v = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (v >= n) return;
    mask_new[(size_t)v * Bp + tile * 32 + lane] = mask_old[(size_t)v * Bp + src[tile * 32 + lane]];
}

}  // namespace afs
