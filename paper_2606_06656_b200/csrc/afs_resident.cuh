// afs_resident.cuh -- the tile-resident PGD kernel: ONE launch runs every PGD iteration (S1..S10) of afs_pgd_run.
//
// Restarts are independent, so a tile of 32 restarts never needs anything from another tile.
// A thread-block cluster of C CTAs owns one tile for the whole run:
//   * every CTA keeps the iterate X_t of the tile in shared memory, X[n][32] (lane <-> restart: every gather is one
//     conflict-free 128-byte LDS, the index/sign words are warp-uniform); what is left of the 227 KB holds the pmf
//     buffers of the EK / CARD bodies (one per warp that may take such a constraint),
//   * the work of an iteration is split over the C CTAs: the materialising ("push") constraints, the bit-parallel
//     counts of the pull clauses and the variables (pull gradients, S6 reduction, step) each by a static partition
//     made at afs_problem_create, and taken warp by warp from one shared work counter inside the CTA,
//   * the pieces meet through L2: per-literal gradients of the push constraints (scratch[tile][slot][32]), the pull
//     gradients (G[tile][v][32]) and the new iterate (XT[tile][v][32]) are written by the warp that computed them
//     and read by others after a
//     cluster barrier (release / acquire at cluster scope); there is no grid-wide synchronisation and no host
//     round trip,
//   * the satisfied counts of iterate t are integer atomics on sat_hist[t mod 3][b]; cluster rank 0 keeps the best
//     count, its step and its sign bits in shared memory.
// One iteration:  P1 push gradients + counts | P2 pull gradients of the own variables -> G
//                 -- cluster barrier --  best-so-far merge of iterate t (rank 0) | P3 S6 + S7 + S8 for the own
//                 variables -> XT (global)  -- cluster barrier --  P4 reload X_{t+1}, sign words.
// The arithmetic of every constraint body, of the pull loops and of the step is the code the streaming kernels
// run (afs_kernels.cuh); only where the operands live differs.
#pragma once
#include <cooperative_groups.h>

#include "afs_kernels.cuh"

namespace afs {

namespace cg = cooperative_groups;

constexpr int RES_WARPS = 32;
constexpr int RES_VCH = 1;   // variables per work item (measured on configs[1]: 1 -> 80.4, 2 -> 84.1, 4 -> 83.1 us/iteration)

template <typename real>
struct XTile {   // x of this lane's restart from the shared tile
    const real* __restrict__ p;   // Xs + lane
    __device__ __forceinline__ real operator()(uint32_t var) const { return p[var * 32u]; }
};
template <typename real>
struct STile {   // scratch[tile][slot][32] in global memory
    real* __restrict__ p;         // scratch + tile * nslots * 32 + lane
    __device__ __forceinline__ void put(int slot, real v) const { p[(size_t)slot * 32] = v; }
    __device__ __forceinline__ real get(int slot) const { return p[(size_t)slot * 32]; }
};

template <typename real>
struct ResArgs {
    int n, steps, C, Bp, ntile;
    int cm_bufs, cm_rows;        // pmf buffers of the CTA (the cm_bufs highest warps own one), rows (cm_maxL + 1) of each
    int meta;                    // bit 0: the rank's small index streams (runs, offsets, push-item literals) are staged
                                 // in shared memory at kernel start; bit 1: its pull words too (cap_words > 0)
    int cap_words, cap_runs, cap_own, cap_plits, cap_cm, cap_push;   // capacities of the staged arrays (max over ranks)
    int64_t nslots;
    const int32_t* pull_ptr;
    const uint32_t* pull_words;
    const int32_t* run_ptr;
    const uint32_t* runs;
    const float* gconst;
    const int32_t* slot_ptr;
    const MedCon* med;
    const uint32_t* med_lits;
    const int32_t* med_slots;
    const LongCon* cm;
    const uint32_t* cm_lits;
    const int32_t* cm_slots;
    const PullClause* pcp;
    const int32_t* var_begin;    // [C+1]
    const int32_t* item_begin;   // [C+1]
    const ResItem* items;
    const int32_t* cm_begin;     // [C+1] ranges of cm_items
    const int32_t* cm_items;     // indices into cm, each rank's heaviest first
    const int32_t* pc_begin;     // [C+1]
    real* XT;                    // [ntile][n][32]
    real* G;                     // [ntile][n][32] pull part of the gradient
    real* scratch;               // [ntile][nslots][32]
    real* aux0;                  // [ntile][med_nnz][32] prefix states of the MED bodies
    real* aux1;
    int64_t med_nnz;
    int32_t* sat_hist;           // [3][Bp] ring of count rows (row t mod 3), zeroed at launch
    uint32_t* best_bits;         // [n][ntile]
    int32_t* best_sat;           // [Bp]
    int32_t* best_step;          // [Bp]
    real lr;
    const int8_t* mask;
};

template <typename real>
__device__ __forceinline__ real ld_cg(const real* p) { return __ldcg(p); }

struct ResMed {   // staged MED item: the constraint record and its bucket
    MedCon mc;
    uint32_t code;
};


template <typename real>
__global__ void __launch_bounds__(RES_WARPS * 32, 1) k_resident(const ResArgs<real> a)
{
    extern __shared__ __align__(16) unsigned char res_smem[];
    __shared__ int s_best_sat[32], s_best_step[32];
    __shared__ int s_ctr, s_ctr_cm;
    cg::cluster_group cluster = cg::this_cluster();
    constexpr int NT = RES_WARPS * 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int rank = (int)(blockIdx.x % (unsigned)a.C), tile = (int)(blockIdx.x / (unsigned)a.C);
    const int n = a.n;
    real* Xs = reinterpret_cast<real*>(res_smem);                       // [n][32]
    uint32_t* S = reinterpret_cast<uint32_t*>(Xs + (size_t)n * 32);      // [n] sign words of X_t
    uint32_t* bestb = S + n;                                            // [n] sign words of the best iterate (rank 0)
    uint2* sbuf0 = reinterpret_cast<uint2*>(S + ((2 * n + 3) & ~3));     // 16-byte aligned
    uint2* sbuf = sbuf0 + warp * PULL_SBUF;
    real* qbase = reinterpret_cast<real*>(sbuf0 + RES_WARPS * PULL_SBUF);
    // pmf buffers belong to the highest warp ids, three per scheduler when there are twelve (the EK / CARD items are
    // the longest dependent chains of the iteration; which warp ids own them made no measurable difference)
    const int cmw = RES_WARPS - 1 - warp;
    real* qcol = qbase + (size_t)(cmw < a.cm_bufs ? cmw : 0) * a.cm_rows * 32 + lane;
    // staged index streams of this rank (a.meta): pull words and runs of the own variables, their stream offsets,
    // literal words / slot ids / records of the own push items
    uint32_t* smw = reinterpret_cast<uint32_t*>(qbase + (size_t)a.cm_bufs * a.cm_rows * 32);
    uint32_t* smr = smw + a.cap_words;
    int32_t* smpp = reinterpret_cast<int32_t*>(smr + a.cap_runs);
    int32_t* smrp = smpp + a.cap_own + 1;
    uint32_t* sml = reinterpret_cast<uint32_t*>(smrp + a.cap_own + 1);
    int32_t* sms = reinterpret_cast<int32_t*>(sml + a.cap_plits);
    int32_t* smo = sms + a.cap_plits;                                   // [cap_cm + cap_push + 1] offsets into sml / sms
    LongCon* smcm = reinterpret_cast<LongCon*>(smo + a.cap_cm + a.cap_push + 1);
    ResMed* smmed = reinterpret_cast<ResMed*>(smcm + a.cap_cm);
    real* XTt = a.XT + (size_t)tile * n * 32 + lane;
    real* Gt = a.G + (size_t)tile * n * 32 + lane;
    const XTile<real> xl{Xs + lane};
    const STile<real> sw{a.scratch + (size_t)tile * a.nslots * 32 + lane};
    const STile<real> ax0{a.aux0 + (size_t)tile * a.med_nnz * 32 + lane}, ax1{a.aux1 + (size_t)tile * a.med_nnz * 32 + lane};
    const ColShared<real> xcol{(uint32_t)__cvta_generic_to_shared(Xs + lane)};
    const int vb = a.var_begin[rank], ve = a.var_begin[rank + 1];
    const int ib = a.item_begin[rank], n_push = a.item_begin[rank + 1] - ib;
    const int mb = a.cm_begin[rank], n_cm = a.cm_begin[rank + 1] - mb;
    const int cb = a.pc_begin[rank], ce = a.pc_begin[rank + 1];
    const int n_cnt = (ce - cb + 31) >> 5;
    const int n_var = (ve - vb + RES_VCH - 1) / RES_VCH;
    const int b = tile * 32 + lane;
    const real one = real(1);

    // base-adjusted views: indexed with the global (absolute) offsets whether staged or not
    const uint32_t* words_v = a.pull_words;
    const uint32_t* runs_v = a.runs;
    const int32_t* pp_v = a.pull_ptr;
    const int32_t* rp_v = a.run_ptr;
    if (a.meta) {
        const int wbase = a.pull_ptr[vb], wn = a.pull_ptr[ve] - wbase + 32;   // + the slack a staged chunk may read
        const int rbase = a.run_ptr[vb], rn = a.run_ptr[ve] - rbase;
        if (a.meta & 2)
            for (int i = tid; i < wn; i += NT) smw[i] = a.pull_words[wbase + i];
        for (int i = tid; i < rn; i += NT) smr[i] = a.runs[rbase + i];
        for (int i = tid; i <= ve - vb; i += NT) { smpp[i] = a.pull_ptr[vb + i]; smrp[i] = a.run_ptr[vb + i]; }
        for (int i = tid; i < n_cm; i += NT) { const LongCon lc = a.cm[a.cm_items[mb + i]]; smcm[i] = lc; smo[i + 1] = lc.L; }
        for (int i = tid; i < n_push; i += NT) {
            const ResItem it = a.items[ib + i];
            ResMed rm; rm.mc = a.med[it.idx]; rm.code = it.code;
            smmed[i] = rm; smo[n_cm + i + 1] = rm.mc.L;
        }
        __syncthreads();
        if (tid == 0) {
            int off = 0;
            smo[0] = 0;
            for (int i = 1; i <= n_cm + n_push; ++i) { off += smo[i]; smo[i] = off; }
        }
        __syncthreads();
        for (int i = warp; i < n_cm + n_push; i += RES_WARPS) {
            const int o = smo[i], L = smo[i + 1] - o;
            const uint32_t* gl = i < n_cm ? a.cm_lits + smcm[i].off : a.med_lits + smmed[i - n_cm].mc.off;
            const int32_t* gs = i < n_cm ? a.cm_slots + smcm[i].off : a.med_slots + smmed[i - n_cm].mc.off;
            for (int j = lane; j < L; j += 32) { sml[o + j] = gl[j]; sms[o + j] = gs[j]; }
        }
        if (a.meta & 2) words_v = smw - wbase;
        runs_v = smr - rbase; pp_v = smpp - vb; rp_v = smrp - vb;
    }
    // P3 takes the own variables vb + warp + RES_WARPS * k; lane k keeps the slot range and the mask of the k-th one
    const int p3_n = ve - vb > warp ? (ve - vb - warp + RES_WARPS - 1) / RES_WARPS : 0;
    const bool p3_regs = ve - vb <= 32 * RES_WARPS;
    int p3_s0 = 0, p3_s1 = 0, p3_mk = 0;
    if (p3_regs && lane < p3_n) {
        const int v = vb + warp + RES_WARPS * lane;
        p3_s0 = a.slot_ptr[v]; p3_s1 = a.slot_ptr[v + 1]; p3_mk = a.mask ? a.mask[v] : 0;
    }
    for (int i = lane; i < PULL_SBUF; i += 32) sbuf[i] = make_uint2(0u, 0u);
    for (int v = warp; v < n; v += RES_WARPS) {
        const real x = ld_cg(XTt + (size_t)v * 32);
        Xs[v * 32 + lane] = x;
        const unsigned sb = __ballot_sync(FULL, x < real(0));
        if (lane == 0) { S[v] = sb; bestb[v] = 0u; }
    }
    if (tid < 32) { s_best_sat[tid] = -1; s_best_step[tid] = 0; }
    if (tid == 0) { s_ctr = 0; s_ctr_cm = 0; }
    __syncthreads();

    for (int t = 0;; ++t) {
        const bool last = t == a.steps;
        // ---- P1 + P2: work items of this CTA, taken from the shared counter (heaviest first)
        {
            int satcnt = 0;
            const int total = n_push + n_cnt + (last ? 0 : n_var);
            if (cmw < a.cm_bufs) {   // EK / CARD constraints first (the heaviest items), by the warps that own a pmf buffer
                for (;;) {
                    int it = 0;
                    if (lane == 0) it = atomicAdd(&s_ctr_cm, 1);
                    it = __shfl_sync(FULL, it, 0);
                    if (it >= n_cm) break;
                    real fe;
                    const LongCon lc = a.meta ? smcm[it] : a.cm[a.cm_items[mb + it]];
                    const uint32_t* lw = a.meta ? sml + smo[it] : a.cm_lits + lc.off;
                    const int32_t* ls = a.meta ? sms + smo[it] : a.cm_slots + lc.off;
                    const unsigned served = cm_body_small<real>(lc, lw, ls, xl, sw, qcol, a.cm_rows, satcnt, fe, false);
                    if (served != FULL) cm_body<real>(lc, lw, ls, xl, sw, qcol, satcnt, fe, false, !((served >> lane) & 1u));
                }
            }
            for (;;) {
                int it = 0;
                if (lane == 0) it = atomicAdd(&s_ctr, 1);
                it = __shfl_sync(FULL, it, 0);
                if (it >= total) break;
                if (it < n_push) {
                    ResMed rm;
                    if (a.meta) rm = smmed[it];
                    else { const ResItem ri = a.items[ib + it]; rm.mc = a.med[ri.idx]; rm.code = ri.code; }
                    const uint32_t* lw = a.meta ? sml + smo[n_cm + it] : a.med_lits + rm.mc.off;
                    const int32_t* ls = a.meta ? sms + smo[n_cm + it] : a.med_slots + rm.mc.off;
                    real fe;
                    med_body<real>(rm.mc, lw, ls, xl, sw, ax0, ax1, satcnt, fe);
                } else if (it < n_push + n_cnt) {
                    // S9 of 32 pull clauses, lane <-> clause, bit r of T <-> restart r
                    const int c = cb + (it - n_push) * 32 + lane;
                    uint32_t T = 0u;
                    if (c < ce) {
                        const uint4* rec = reinterpret_cast<const uint4*>(a.pcp + c);
                        const uint4 h0 = rec[0], h1 = rec[1];
                        const uint32_t lit[PULL_MAX_LEN] = {h0.y, h0.z, h0.w, h1.x, h1.y};
                        const int L = (int)(h0.x & 7u), kind = (int)((h0.x >> 3) & 3u);
                        uint32_t vor = 0u, vand = 0xffffffffu, vxor = 0u;
#pragma unroll
                        for (int j = 0; j < PULL_MAX_LEN; ++j)
                            if (j < L) {
                                const uint32_t tj = S[lit[j] & LIT_VAR] ^ ((lit[j] >> 31) ? 0xffffffffu : 0u);
                                vor |= tj; vand &= tj; vxor ^= tj;
                            }
                        const uint32_t par = ((h0.x >> 5) & 1u) ? 0xffffffffu : 0u;
                        T = kind == (int)PH_KIND_OR ? vor : kind == (int)PH_KIND_XOR ? ~(vxor ^ par) : (vor & ~vand);
                    }
                    satcnt += bit_column_sums(T, lane);
                } else {
                    const int i0 = (it - n_push - n_cnt) * RES_VCH;
                    for (int i = i0; i < min(i0 + RES_VCH, ve - vb); ++i) {
                        const int v = vb + i;
                        const int mk = a.mask ? a.mask[v] : 0;
                        real g[1] = {real(0)};
                        if (mk == 0) {
                            g[0] = (real)a.gconst[v];
                            pull_variable<real, 1>(runs_v, rp_v[v], rp_v[v + 1], words_v, pp_v[v], xcol,
                                                   32u * (uint32_t)sizeof(real), lane, sbuf, g);
                        }
                        Gt[(size_t)v * 32] = g[0];
                    }
                }
            }
            if (satcnt) atomicAdd(a.sat_hist + (size_t)(t % 3) * a.Bp + b, satcnt);
        }
        cluster.sync();
        if (tid == 0) { s_ctr = 0; s_ctr_cm = 0; }
        // ---- S10: iterate t against the best so far (rank 0 holds the record of the tile)
        if (rank == 0) {
            const int sp = __ldcg(a.sat_hist + (size_t)(t % 3) * a.Bp + b);
            if (warp == 1) a.sat_hist[(size_t)((t + 1) % 3) * a.Bp + b] = 0;   // the row of the next iterate (ring of three)
            const bool imp = sp > s_best_sat[lane];
            const unsigned impmask = __ballot_sync(FULL, imp);
            if (impmask)
                for (int v = tid; v < n; v += NT) bestb[v] = (bestb[v] & ~impmask) | (S[v] & impmask);
            if (last) {
                __syncthreads();
                if (warp == 0) {
                    a.best_sat[b] = imp ? sp : s_best_sat[lane];
                    a.best_step[b] = imp ? t : s_best_step[lane];
                }
                for (int v = tid; v < n; v += NT) a.best_bits[(size_t)v * a.ntile + tile] = bestb[v];
            }
        }
        if (last) break;
        // ---- P3: S6 (fixed transposed-CSR order) + S7 + S8 for the own variables, two at a time: G and the first
        // four gradient rows of both are requested together (everything here comes from L2), then added in slot order
        for (int k = 0; k < p3_n; k += 2) {
            int v[2], s0[2], s1[2], mk[2];
            bool ok[2];
            real x[2], g[2], pre[2][4];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                ok[h] = k + h < p3_n;
                const int kk = ok[h] ? k + h : k;
                v[h] = vb + warp + RES_WARPS * kk;
                if (p3_regs) {
                    s0[h] = __shfl_sync(FULL, p3_s0, kk); s1[h] = __shfl_sync(FULL, p3_s1, kk); mk[h] = __shfl_sync(FULL, p3_mk, kk);
                } else {
                    s0[h] = a.slot_ptr[v[h]]; s1[h] = a.slot_ptr[v[h] + 1]; mk[h] = a.mask ? a.mask[v[h]] : 0;
                }
                if (mk[h] != 0) s1[h] = s0[h];
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                x[h] = Xs[v[h] * 32 + lane];
                g[h] = ld_cg(Gt + (size_t)v[h] * 32);
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    pre[h][i] = s0[h] + i < s1[h] ? ld_cg(sw.p + (size_t)(s0[h] + i) * 32) : real(0);
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (!ok[h]) continue;
                const real* __restrict__ sc = sw.p;
                int s = s0[h];
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    if (s + i < s1[h]) g[h] += pre[h][i];
                s += 4;
                for (; s + 4 <= s1[h]; s += 4) {
                    real g0 = ld_cg(sc + (size_t)s * 32), g1 = ld_cg(sc + (size_t)(s + 1) * 32);
                    real g2 = ld_cg(sc + (size_t)(s + 2) * 32), g3 = ld_cg(sc + (size_t)(s + 3) * 32);
                    g[h] += g0; g[h] += g1; g[h] += g2; g[h] += g3;
                }
                for (; s < s1[h]; ++s) g[h] += ld_cg(sc + (size_t)s * 32);
                real xn = x[h] - a.lr * g[h];
                xn = xn > one ? one : xn;
                xn = xn < -one ? -one : xn;
                if (mk[h] != 0) xn = x[h];
                XTt[(size_t)v[h] * 32] = xn;
            }
        }
        cluster.sync();
        // ---- P4: the record of iterate t, then X_{t+1} and its sign words
        if (rank == 0 && warp == 0) {
            const int sp = __ldcg(a.sat_hist + (size_t)(t % 3) * a.Bp + b);
            if (sp > s_best_sat[lane]) { s_best_sat[lane] = sp; s_best_step[lane] = t; }
        }
#pragma unroll 8
        for (int v = warp; v < n; v += RES_WARPS) {
            const real x = ld_cg(XTt + (size_t)v * 32);
            Xs[v * 32 + lane] = x;
            const unsigned sb = __ballot_sync(FULL, x < real(0));
            if (lane == 0) S[v] = sb;
        }
        __syncthreads();
    }
}

// X[B,n] -> XT[tile][v][32] with the mask applied at entry; -0.0 -> +0.0 (G13)
template <typename real>
__global__ void __launch_bounds__(256) k_res_in(const real* __restrict__ X, real* __restrict__ XT, int B, int n,
                                                const int8_t* __restrict__ mask)
{
    __shared__ real tile[32][33];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int v0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
    for (int r = ty; r < 32; r += 8) {   // columns behind the batch: copies of the last restart (see k_transpose_in)
        int b = min(b0 + r, B - 1), v = v0 + tx;
        real x = real(0);
        if (v < n) x = X[(size_t)b * n + v] + real(0);
        tile[r][tx] = x;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        int v = v0 + r, b = b0 + tx;
        if (v < n) {
            real x = tile[tx][r];
            if (mask) { int mk = mask[v]; if (mk != 0) x = mk > 0 ? real(1) : real(-1); }
            XT[((size_t)blockIdx.y * n + v) * 32 + tx] = x;
        }
    }
}

// XT[tile][v][32], best_bits[n][ntile] -> X[B,n], best_assign[B,n]; best_sat / best_step copied out
template <typename real>
__global__ void __launch_bounds__(256) k_res_out(const real* __restrict__ XT, const uint32_t* __restrict__ best_bits,
                                                 const int32_t* __restrict__ bsat, const int32_t* __restrict__ bstep,
                                                 int B, int n, int ntile, real* __restrict__ X,
                                                 int8_t* __restrict__ best_assign, int32_t* __restrict__ best_sat,
                                                 int32_t* __restrict__ best_step)
{
    __shared__ real tile[32][33];
    __shared__ unsigned s_bits[32];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int v0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
    for (int r = ty; r < 32; r += 8) {
        int v = v0 + r;
        tile[r][tx] = v < n ? XT[((size_t)blockIdx.y * n + v) * 32 + tx] : real(0);
        if (tx == 0) s_bits[r] = v < n ? best_bits[(size_t)v * ntile + blockIdx.y] : 0u;
    }
    __syncthreads();
    for (int r = ty; r < 32; r += 8) {
        int bb = b0 + r, v = v0 + tx;
        if (bb < B && v < n) {
            if (X) X[(size_t)bb * n + v] = tile[tx][r];
            if (best_assign) best_assign[(size_t)bb * n + v] = ((s_bits[tx] >> r) & 1u) ? -1 : 1;
        }
    }
    if (blockIdx.x == 0 && ty == 0 && b0 + tx < B) {
        if (best_sat) best_sat[b0 + tx] = bsat[b0 + tx];
        if (best_step) best_step[b0 + tx] = bstep[b0 + tx];
    }
}

// dynamic shared memory of k_resident for n variables and cm_bufs pmf buffers of cm_rows rows (without staged streams)
template <typename real>
inline size_t res_smem_bytes(int n, int cm_bufs, int cm_rows)
{
    return (size_t)n * 32 * sizeof(real) + (size_t)((2 * n + 3) & ~3) * 4 + (size_t)RES_WARPS * PULL_SBUF * sizeof(uint2) +
           (size_t)cm_bufs * cm_rows * 32 * sizeof(real);
}
// bytes of the staged index streams of one rank, capacities as in ResArgs
inline size_t res_meta_bytes(int cap_words, int cap_runs, int cap_own, int cap_plits, int cap_cm, int cap_push)
{
    return 4 * ((size_t)cap_words + cap_runs + 2 * ((size_t)cap_own + 1) + 2 * (size_t)cap_plits + cap_cm + cap_push + 1) +
           sizeof(LongCon) * (size_t)cap_cm + sizeof(ResMed) * (size_t)cap_push + 16;
}

}  // namespace afs
