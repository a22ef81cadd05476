// afs_run.cuh -- launch orchestration of the device entry points of include/afs.h, templated on the arithmetic type;
// instantiated by afs_f32.cu (the product) and afs_f64.cu (the fp64 verification build).
// Streaming path: per PGD step one launch per non-empty push bucket (medium / long constraints) plus one fused
// variable pass; no host round trip inside the loop (everything is enqueued on the caller's stream).
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdio>

#include "afs_kernels.cuh"
#include "afs_resident.cuh"
#include "afs_gm.cuh"
#include "afs_launch.h"

namespace afs {

static int var_grid_x(int n) { return (n + VAR_WARPS * VAR_VPW - 1) / (VAR_WARPS * VAR_VPW); }

// variable pass: as many 32-restart sub-tiles per lane as the batch allows (4, 2 or 1)
template <typename real, bool EVAL, bool LONGT, bool CONV>
static void launch_var_l(const VarArgs<real>& a, int gx, int tiles, cudaStream_t st)
{
    if (sizeof(real) == 4 && tiles % 4 == 0) k_var<real, EVAL, 4, LONGT, CONV><<<dim3(gx, tiles / 4), VAR_WARPS * 32, 0, st>>>(a);
    else if (tiles % 2 == 0) k_var<real, EVAL, 2, LONGT, CONV><<<dim3(gx, tiles / 2), VAR_WARPS * 32, 0, st>>>(a);
    else k_var<real, EVAL, 1, LONGT, CONV><<<dim3(gx, tiles), VAR_WARPS * 32, 0, st>>>(a);
}
template <typename real, bool EVAL, bool LONGT>
static void launch_var_c(const VarArgs<real>& a, int gx, int tiles, cudaStream_t st)
{
    if (!EVAL && (a.tol > real(0) || a.maskT)) launch_var_l<real, EVAL, LONGT, !EVAL>(a, gx, tiles, st);
    else launch_var_l<real, EVAL, LONGT, false>(a, gx, tiles, st);
}
template <typename real, bool EVAL>
static void launch_var(afs_problem* P, VarArgs<real>& a, int gx, int tiles, const RunState* rs, cudaStream_t st)
{
    if (P->n_long > 0) {   // the LONG class's share first (k_glong), from the pairs and rows the long kernels just wrote
        real* GL = (real*)P->ws.GL;
        {
            ProfSpan span(P, 6, st);
            const real* lrows = a.scratch + (size_t)P->nslots_a * a.Bp;
            const int nl = (int)(P->nslots - P->nslots_a);
            const int8_t* mk = EVAL ? nullptr : a.mask;
            if (tiles % 2 == 0) {
                const long long warps = (long long)P->n * (tiles / 2);
                k_glong<real, 2><<<(unsigned)std::min<long long>((warps + 7) / 8, (long long)P->sm_count * 16), 256, 0, st>>>(P->n, tiles, a.Bp, P->d_lslot_ptr, P->d_lslot_info,
                                                                            a.Xin, lrows, nl, (const real*)P->ws.bnd, mk, GL, rs);
            } else {
                const long long warps = (long long)P->n * tiles;
                k_glong<real, 1><<<(unsigned)std::min<long long>((warps + 7) / 8, (long long)P->sm_count * 16), 256, 0, st>>>(P->n, tiles, a.Bp, P->d_lslot_ptr, P->d_lslot_info,
                                                                            a.Xin, lrows, nl, (const real*)P->ws.bnd, mk, GL, rs);
            }
        }
        a.GL = GL;
        launch_var_c<real, EVAL, true>(a, gx, tiles, st);
    } else {
        launch_var_c<real, EVAL, false>(a, gx, tiles, st);
    }
}

// ----------------------------------------------------------------------------------------------------------------
// push phase: gradients of the medium and long constraints of iterate XT into scratch (+ counts, + FE)
// ----------------------------------------------------------------------------------------------------------------
template <typename real>
static afs_status launch_push(afs_problem* P, const real* XT, const uint32_t* Sw, const uint32_t* SATw, int Bp,
                              real* scratch, int32_t* sat, real* fe_med, real* fe_cm, real* fe_long, const RunState* rs,
                              cudaStream_t st)
{
    const int tiles = Bp / 32;
    if (P->n_cm > 0) {
        const int c0 = 0, c1 = (int)P->n_cm;
        int gx = (c1 - c0 + 3) / 4;
        int cap = (P->sm_count * 16 + tiles - 1) / tiles;
        if (gx > cap) gx = cap < 1 ? 1 : cap;
        const int qrows = P->cm_maxL + 1;
        const size_t smem = (size_t)4 * qrows * 32 * sizeof(real);
        // kernel attributes are per device and per instantiation: set before every launch (cheap), never cached
        if (smem > 48 * 1024)
            CU(cudaFuncSetAttribute(k_cmed<real>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        ProfSpan span(P, 3, st);
        k_cmed<real><<<dim3(gx, tiles), 128, smem, st>>>((P->unit_w_mode && P->d_cm_u) ? P->d_cm_u : P->d_cm, c0, c1, P->d_cm_lits, P->d_cm_slots, XT, Bp, scratch, sat,
                                                        fe_cm, qrows, rs);
        P->last_launches++;
    }
    if (P->n_med > 0) {
        int gx = ((int)P->n_med + 3) / 4;
        int cap = (P->sm_count * 16 + tiles - 1) / tiles;   // enough CTAs to fill the chip, grid-stride beyond
        if (gx > cap) gx = cap < 1 ? 1 : cap;
        ProfSpan span(P, 4, st);
        k_med<real><<<dim3(gx, tiles), 128, 0, st>>>((P->unit_w_mode && P->d_med_u) ? P->d_med_u : P->d_med, 0, (int)P->n_med, P->d_med_lits, P->d_med_slots, XT, Bp, scratch,
                                                    (real*)P->ws.aux[0], (real*)P->ws.aux[1], sat, fe_med, rs);
        P->last_launches++;
    }
    if (P->n_long > 0) return launch_long_all<real>(P, XT, Sw, SATw, Bp, scratch, sat, fe_long, rs, st);
    return AFS_OK;
}

template <typename real>
static afs_status launch_count(afs_problem* P, const real* XT, int Bp, int32_t* sat, const RunState* rs, cudaStream_t st)
{
    CU(cudaMemsetAsync(sat, 0, (size_t)Bp * sizeof(int32_t), st));
    if (P->m > 0) {
        const int tiles = Bp / 32;
        int gx = (P->m + 7) / 8;
        int cap = (P->sm_count * 8 + tiles - 1) / tiles;
        if (gx > cap) gx = cap < 1 ? 1 : cap;
        ProfSpan span(P, 18, st);
        k_count<real><<<dim3(gx, tiles), 256, 0, st>>>(P->d_count, P->d_count_lits, P->m, XT, Bp, sat, rs);
        P->last_launches++;
    }
    return AFS_OK;
}

// ----------------------------------------------------------------------------------------------------------------
template <typename real>
static afs_status eval_grad_impl(afs_problem* P, const real* X, int32_t B, real* F, real* G, void* stream)
{
    DeviceScope dev_scope(P);
    afs_status s = enter(P, B);
    if (s != AFS_OK) return s;
    if (!X) return AFS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int Bp = ((B + 31) / 32) * 32;
    if ((s = ensure_workspace(P, Bp, sizeof(real), 2)) != AFS_OK) return s;
    if ((s = ensure_eval_buffers(P, Bp, sizeof(real))) != AFS_OK) return s;
    Workspace& w = P->ws;
    const int wBp = Bp;   // kernels run on the first Bp columns with row stride Bp
    real* XT = (real*)w.XT[0];
    real* GT = (real*)w.XT[1];
    real* scratch = (real*)w.scratch;
    real* fe_med = (real*)w.fe_med; real* fe_long = (real*)w.fe_long; real* fe_cm = (real*)w.fe_cm;
    real* fpart = (real*)w.f_part;
    dim3 tg((P->n + 31) / 32, Bp / 32);
    k_transpose_in<real><<<tg, 256, 0, st>>>(X, XT, B, P->n, wBp, nullptr, w.S[0], w.SAT[0]);
    P->last_launches++;
    if ((s = launch_push<real>(P, XT, w.S[0], w.SAT[0], wBp, scratch, nullptr, fe_med, fe_cm, fe_long, nullptr, st)) != AFS_OK) return s;
    VarArgs<real> a{};
    a.n = P->n; a.Bp = wBp; a.t = 0;
    a.pull_ptr = P->d_pull_ptr; a.pull_words = P->d_pull_words; a.run_ptr = P->d_run_ptr; a.runs = P->d_runs;
    a.gconst = P->d_pull_gconst; a.slot_ptr = P->d_slot_ptr;
    a.scratch = scratch; a.Xin = XT; a.Xout = nullptr; a.lr = real(0); a.mask = nullptr;
    a.GT = GT;
    const int gx = var_grid_x(P->n);
    if (G) {
        launch_var<real, true>(P, a, gx, Bp / 32, nullptr, st);
        P->last_launches++;
    }
    if (F) {
        const int fgx = fe_pull_grid_x(P);
        k_fe_pull<real><<<dim3(fgx, Bp / 32), 256, 0, st>>>(P->d_pc, P->d_pc_lits, (int)P->n_pull, XT, wBp, fpart);
        k_reduce_F<real><<<(B + 127) / 128, 128, 0, st>>>(fpart, fgx * 8, fe_med, (int)P->n_med, fe_cm, (int)P->n_cm,
                                                         fe_long, (int)P->n_long, wBp, B, F);
        P->last_launches += 2;
    }
    if (G) {
        k_transpose_out<real><<<tg, 256, 0, st>>>(GT, G, B, P->n, wBp);
        P->last_launches++;
    }
    CU(cudaGetLastError());
    return AFS_OK;
}

// per-constraint gradient magnitudes (afs_gm.cuh): one evaluation with unit weights, then a reduction per class
template <typename real>
static afs_status grad_l1_impl(afs_problem* P, const real* X, int32_t B, real* gm, void* stream)
{
    DeviceScope dev_scope(P);
    afs_status s = enter(P, B);
    if (s != AFS_OK) return s;
    if (!X || !gm) return AFS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int Bp = ((B + 31) / 32) * 32, ntile = Bp / 32;
    if ((s = ensure_workspace(P, Bp, sizeof(real), 3)) != AFS_OK) return s;
    if ((s = ensure_eval_buffers(P, Bp, sizeof(real))) != AFS_OK) return s;
    Workspace& w = P->ws;
    const int64_t need = (int64_t)(P->m > 0 ? P->m : 1) * (w.Bp / 32) * 8;
    if (w.gm_elems < need) {
        CU(cudaDeviceSynchronize());
        if (w.gm_part) cudaFree(w.gm_part);
        w.gm_part = nullptr; w.gm_elems = 0;
        if (cudaMalloc(&w.gm_part, (size_t)need) != cudaSuccess) { (void)cudaGetLastError(); return AFS_ERR_ALLOC; }
        w.gm_elems = need; w.bytes += (size_t)need;
    }
    real* XT = (real*)w.XT[0];
    real* scratch = (real*)w.scratch;
    real* part = (real*)w.gm_part;
    dim3 tg((P->n + 31) / 32, ntile);
    k_transpose_in<real><<<tg, 256, 0, st>>>(X, XT, B, P->n, Bp, nullptr, w.S[0], w.SAT[0]);
    P->unit_w_mode = true;
    s = launch_push<real>(P, XT, w.S[0], w.SAT[0], Bp, scratch, nullptr, nullptr, nullptr, nullptr, nullptr, st);
    P->unit_w_mode = false;
    if (s != AFS_OK) return s;
    if (P->n_pull > 0)
        k_gm_pull<real><<<dim3((unsigned)((P->n_pull + 3) / 4), ntile), 128, 0, st>>>(P->d_pcp, (int)P->n_pull, P->d_pull_id, XT, Bp, B, part);
    if (P->n_med > 0)
        k_gm_rows<real, MedCon><<<dim3((unsigned)((P->n_med + 3) / 4), ntile), 128, 0, st>>>(P->d_med, (int)P->n_med, P->d_med_slots,
                                                                                           P->d_med_id, scratch, Bp, B, part);
    if (P->n_cm > 0)
        k_gm_rows<real, LongCon><<<dim3((unsigned)((P->n_cm + 3) / 4), ntile), 128, 0, st>>>(P->d_cm, (int)P->n_cm, P->d_cm_slots,
                                                                                           P->d_cm_id, scratch, Bp, B, part);
    if (P->n_long > 0) {
        const long long warps = (long long)P->n_long * ntile;
        k_gm_long<real><<<(unsigned)((warps + 3) / 4), 128, 0, st>>>(P->d_long, (int)P->n_long, P->d_long_lits, P->d_long_slots,
                                                                   P->d_long_id, w.S[0], w.SAT[0], ntile, Bp, B,
                                                                   scratch + (size_t)P->nslots_a * Bp, (int)P->nslots_a,
                                                                   (int)(P->nslots - P->nslots_a), (const real*)w.bnd, part);
    }
    if (P->m > 0) k_gm_final<real><<<(P->m + 255) / 256, 256, 0, st>>>(part, P->m, ntile, gm);
    P->last_launches += 6;
    CU(cudaGetLastError());
    return AFS_OK;
}

template <typename real>
static afs_status round_count_impl(afs_problem* P, const real* X, int32_t B, int8_t* assign, int32_t* sat, void* stream)
{
    DeviceScope dev_scope(P);
    afs_status s = enter(P, B);
    if (s != AFS_OK) return s;
    if (!X || !sat) return AFS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int Bp = ((B + 31) / 32) * 32;
    if ((s = ensure_workspace(P, Bp, sizeof(real), 2)) != AFS_OK) return s;
    Workspace& w = P->ws;
    real* XT = (real*)w.XT[0];
    dim3 tg((P->n + 31) / 32, Bp / 32);
    k_transpose_in<real><<<tg, 256, 0, st>>>(X, XT, B, P->n, Bp, nullptr, nullptr, nullptr);
    P->last_launches++;
    if ((s = launch_count<real>(P, XT, Bp, w.sat_hist, nullptr, st)) != AFS_OK) return s;
    CU(cudaMemcpyAsync(sat, w.sat_hist, (size_t)B * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
    if (assign) {
        k_assign_out<real><<<tg, 256, 0, st>>>(XT, assign, B, P->n, Bp);
        P->last_launches++;
    }
    CU(cudaGetLastError());
    return AFS_OK;
}

// ----------------------------------------------------------------------------------------------------------------
// tile-resident path: one launch for the whole run.  Eligible when no constraint needs the CTA-cooperative LONG
// kernel and the tile X[n][32] plus the rank's gradient rows fit the 227 KB of shared memory.
// ----------------------------------------------------------------------------------------------------------------
constexpr size_t RES_SMEM_MAX = 227 * 1024 - 512;

// Shared-memory layout of one CTA of the resident kernel for plan pi: the tile and its sign words always; then, as far
// as the 227 KB go and in this order: the rank's small index streams (runs, stream offsets, literals of its push
// items), pmf buffers for the EK / CARD bodies -- up to 12, or one per constraint of the rank if that is fewer: the
// warps that own one carry the longest dependent chains of the iteration and must not be few -- and last the rank's
// pull words (the largest stream; 32 warps hide its L2 latency when it stays in global memory).
struct ResLayout { bool ok; int cm_bufs; int meta; int cap_words; size_t bytes; };
template <typename real>
static ResLayout resident_layout(const afs_problem* P, int pi)
{
    const ResPlan& rp = P->res[pi];
    size_t used = res_smem_bytes<real>(P->n, 0, 0);
    if (used > RES_SMEM_MAX) return {false, 0, 0, 0, 0};
    const size_t per = P->n_cm > 0 ? (size_t)(P->cm_maxL + 1) * 32 * sizeof(real) : 0;
    if (per != 0 && used + per > RES_SMEM_MAX) return {false, 0, 0, 0, 0};
    int meta = 0, nb = 0, cap_words = 0;
    const size_t small = res_meta_bytes(0, rp.cap_runs, rp.cap_own, rp.cap_plits, rp.cap_cm, rp.cap_push);
    if (used + small + per <= RES_SMEM_MAX) { meta = 1; used += small; }
    if (per != 0) {
        const int want = std::min(RES_WARPS, std::min(12, std::max(rp.cap_cm, 1)));
        nb = (int)std::min<size_t>((size_t)want, (RES_SMEM_MAX - used) / per);
        used += (size_t)nb * per;
    }
    if (meta && used + 4 * (size_t)rp.cap_words <= RES_SMEM_MAX) { meta |= 2; cap_words = rp.cap_words; used += 4 * (size_t)cap_words; }
    if (per != 0 && nb < RES_WARPS) {   // what is left goes to more pmf buffers
        const int more = (int)std::min<size_t>((size_t)(RES_WARPS - nb), (RES_SMEM_MAX - used) / per);
        nb += more; used += (size_t)more * per;
    }
    return {true, nb, meta, cap_words, used};
}

template <typename real>
static int resident_plan(const afs_problem* P, int ntile)
{
    if (P->n_long > 0 || !P->res[0].d_var_begin) return -1;
    int pi = RES_PLANS - 1;   // plan pi: pi + 1 CTAs per tile; the largest cluster size whose CTAs are all resident at once
    while (pi > 0 && (long long)ntile * (pi + 1) > P->sm_count) --pi;
    return resident_layout<real>(P, pi).ok ? pi : -1;
}

template <typename real>
static afs_status pgd_run_resident(afs_problem* P, int pi, real* X, int32_t B, int32_t steps, real lr,
                                   const int8_t* mask, int8_t* best_assign, int32_t* best_sat, int32_t* best_step,
                                   cudaStream_t st)
{
    Workspace& w = P->ws;
    const int Bp = ((B + 31) / 32) * 32, ntile = Bp / 32;
    const ResPlan& rp = P->res[pi];
    real* XT = (real*)w.XT[0];
    dim3 tg((P->n + 31) / 32, ntile);
    k_res_in<real><<<tg, 256, 0, st>>>(X, XT, B, P->n, mask);
    CU(cudaMemsetAsync(w.sat_hist, 0, (size_t)3 * Bp * sizeof(int32_t), st));
    ResArgs<real> a{};
    a.n = P->n; a.steps = steps; a.C = rp.C; a.Bp = Bp; a.ntile = ntile; a.nslots = P->nslots;
    const ResLayout lay = resident_layout<real>(P, pi);
    a.cm_bufs = lay.cm_bufs; a.cm_rows = P->cm_maxL + 1; a.meta = lay.meta;
    a.cap_words = lay.cap_words; a.cap_runs = rp.cap_runs; a.cap_own = rp.cap_own; a.cap_plits = rp.cap_plits;
    a.cap_cm = rp.cap_cm; a.cap_push = rp.cap_push;
    a.cm_begin = rp.d_cm_begin; a.cm_items = rp.d_cm_items;
    a.G = (real*)w.XT[1];
    a.aux0 = (real*)w.aux[0]; a.aux1 = (real*)w.aux[1]; a.med_nnz = P->med_nnz;
    a.pull_ptr = P->d_pull_ptr; a.pull_words = P->d_pull_words; a.run_ptr = P->d_run_ptr; a.runs = P->d_runs;
    a.gconst = P->d_pull_gconst; a.slot_ptr = P->d_slot_ptr;
    a.med = P->d_med; a.med_lits = P->d_med_lits; a.med_slots = P->d_med_slots;
    a.cm = P->d_cm; a.cm_lits = P->d_cm_lits; a.cm_slots = P->d_cm_slots;
    a.pcp = P->d_pcp;
    a.var_begin = rp.d_var_begin; a.item_begin = rp.d_item_begin; a.items = rp.d_items; a.pc_begin = rp.d_pc_begin;
    a.XT = XT; a.scratch = (real*)w.scratch; a.sat_hist = w.sat_hist;
    a.best_bits = w.best_bits[0]; a.best_sat = w.best_sat[0]; a.best_step = w.best_step[0];
    a.lr = lr; a.mask = mask;
    const size_t smem = lay.bytes;
    CU(cudaFuncSetAttribute(k_resident<real>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RES_SMEM_MAX));
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)(ntile * rp.C));
    cfg.blockDim = dim3(RES_WARPS * 32);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)rp.C; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    P->prof.on = P->prof.stride > 0;
    {
        ProfSpan span(P, 0, st);
        CU(cudaLaunchKernelEx(&cfg, k_resident<real>, a));
    }
    P->prof.on = false;
    k_res_out<real><<<tg, 256, 0, st>>>(XT, w.best_bits[0], w.best_sat[0], w.best_step[0], B, P->n, ntile, X, best_assign,
                                        best_sat, best_step);
    P->last_launches += 3;
    P->last_resident = 1;
    CU(cudaGetLastError());
    return AFS_OK;
}

template <typename real>
static afs_status pgd_run_impl(afs_problem* P, real* X, int32_t B, int32_t steps, real lr, const int8_t* mask,
                               int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* stream,
                               real tol = real(0), int32_t* conv_step = nullptr, bool per_restart_masks = false)
{
    DeviceScope dev_scope(P);
    afs_status s = enter(P, B);
    if (s != AFS_OK) return s;
    if (!X || steps < 0 || !std::isfinite((double)lr)) return AFS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int Bp = ((B + 31) / 32) * 32;
    // convergence detection (tol > 0) lives in the streaming path, where stopped restarts are retired
    const int plan = (P->opt_mode == 1 || tol > real(0) || per_restart_masks) ? -1 : resident_plan<real>(P, Bp / 32);
    if (per_restart_masks && !mask) return AFS_ERR_INVALID_ARG;
    if (P->opt_mode == 2 && plan < 0) return AFS_ERR_UNSUPPORTED;
    // count rows: a ring of three on both paths (memory does not grow with the number of steps)
    if ((s = ensure_workspace(P, Bp, sizeof(real), 3)) != AFS_OK) return s;
    Workspace& w = P->ws;
    if (per_restart_masks && w.maskT_elems < (int64_t)P->n * w.Bp) {
        CU(cudaDeviceSynchronize());
        if (w.maskT) cudaFree(w.maskT);
        w.maskT = nullptr; w.maskT_elems = 0;
        // two copies: a compaction gathers the masks of the active restarts from one into the other
        if (cudaMalloc((void**)&w.maskT, (size_t)2 * P->n * w.Bp) != cudaSuccess) { (void)cudaGetLastError(); return AFS_ERR_ALLOC; }
        w.maskT_elems = (int64_t)P->n * w.Bp;
        w.bytes += (size_t)2 * P->n * w.Bp;
    }
    P->last_resident = 0;
    if (plan >= 0) return pgd_run_resident<real>(P, plan, X, B, steps, lr, mask, best_assign, best_sat, best_step, st);
    real* XT[3] = {(real*)w.XT[0], (real*)w.XT[1], (real*)w.XT[2]};
    real* scratch = (real*)w.scratch;
    const int tiles = Bp / 32;
    dim3 tg((P->n + 31) / 32, tiles);
    // buffer roles, tracked here (they rotate at every step and at every compaction)
    int xc = 0;              // XT[xc] = X_t
    int sc_ = 0, sp_ = 1;    // S/SAT[sc_] = words of X_t, S[sp_] = sign words of X_{t-1}
    int bc = 0;              // best_sat/best_step[bc] = record over the iterates merged so far
    int bb = 0;              // best_bits[bb]
    int oc = 0;              // orig[oc]
    bool pending = false;    // iterate t-1 is counted but not merged yet (the variable pass of iteration t merges it)
    RunState* rs = w.rs;
    const bool conv = tol > real(0) || per_restart_masks;   // the extended variable pass (its state must be initialised)
    const int8_t* mask1 = per_restart_masks ? nullptr : mask;   // the one mask shared by all restarts, if that is the mode
    typedef typename DBits<real>::type dbits_t;
    dbits_t* delta = static_cast<dbits_t*>(w.delta);     // [3][Bp], row t % 3 = max |dX| of step t
    bool dpending = false;                               // the last step's row is not folded into conv yet
    int8_t* maskT[2] = {w.maskT, w.maskT ? w.maskT + (size_t)P->n * w.Bp : nullptr};
    int mc = 0;              // maskT[mc] = the per-restart masks in the current column order
    if (conv) {
        launch_fill_i32(w.conv[0], (size_t)Bp, -1, st);
        CU(cudaMemsetAsync(w.delta, 0, (size_t)3 * Bp * sizeof(dbits_t), st));
    }
    k_transpose_in<real><<<tg, 256, 0, st>>>(X, XT[0], B, P->n, Bp, mask, w.S[0], w.SAT[0], per_restart_masks ? P->n : 0,
                                             per_restart_masks ? maskT[0] : nullptr);
    k_run_init<<<(Bp + 255) / 256, 256, 0, st>>>(rs, B, Bp, w.orig[0], w.moved);
    P->last_launches += 2;
    CU(cudaMemsetAsync(w.sat_hist, 0, (size_t)3 * Bp * sizeof(int32_t), st));
    launch_fill_i32(w.best_sat[0], (size_t)Bp, -1, st);
    CU(cudaMemsetAsync(w.best_step[0], 0, (size_t)Bp * sizeof(int32_t), st));
    P->last_launches++;
    const int gx = var_grid_x(P->n);
    if (mask1 && P->n_long > 0 && steps > 0) {   // the fixed variables' literals leave the long constraints for this run
        if ((s = launch_long_fold(P, mask1, st)) != AFS_OK) return s;
    }
    const int K = P->retire_every;   // 0: never
    for (int t = 0; t < steps; ++t) {
        P->prof.on = P->prof.stride > 0 && t % P->prof.stride == 0;
        const bool retire = K > 0 && (t + 1) % K == 0 && t + 1 < steps;
        const real* Xin = XT[xc];
        const int xn = (xc + 1) % 3;
        int32_t* sat_cur = w.sat_hist + (size_t)(t % 3) * Bp;
        if ((s = launch_push<real>(P, Xin, w.S[sc_], w.SAT[sc_], Bp, scratch, sat_cur, nullptr, nullptr, nullptr, rs, st)) != AFS_OK) return s;
        VarArgs<real> a{};
        a.n = P->n; a.Bp = Bp; a.t = t;
        a.pull_ptr = P->d_pull_ptr; a.pull_words = P->d_pull_words; a.run_ptr = P->d_run_ptr; a.runs = P->d_runs;
        a.gconst = P->d_pull_gconst; a.slot_ptr = P->d_slot_ptr;
        a.scratch = scratch; a.Xin = Xin; a.Xout = XT[xn]; a.lr = lr; a.mask = mask1;
        a.maskT = per_restart_masks ? maskT[mc] : nullptr;
        a.sat_prev = pending ? w.sat_hist + (size_t)((t + 2) % 3) * Bp : nullptr;
        a.sat_zero = w.sat_hist + (size_t)((t + 1) % 3) * Bp;
        a.best_sat_in = w.best_sat[bc]; a.best_sat_out = w.best_sat[bc ^ 1];
        a.best_step_in = w.best_step[bc]; a.best_step_out = w.best_step[bc ^ 1];
        a.S_prev = w.S[sp_]; a.S_next = w.S[sp_]; a.SAT_next = w.SAT[sp_]; a.best_bits = w.best_bits[bb];
        a.rs = rs; a.moved = retire ? w.moved : nullptr;
        a.tol = tol;
        if (conv) {
            a.conv_in = w.conv[bc]; a.conv_out = w.conv[bc ^ 1];
            a.delta_prev = dpending ? delta + (size_t)((t + 2) % 3) * Bp : nullptr;
            a.delta_cur = delta + (size_t)(t % 3) * Bp; a.delta_zero = delta + (size_t)((t + 1) % 3) * Bp;
        }
        // S9 of the pull clauses needs only the (complete) sign words of X_t: it runs on the library's second stream
        // beside the variable pass and is joined before anything reads the count row of X_t
        const bool side = P->n_pull > 0;
        if (side) {
            CU(cudaEventRecord(P->ev_fork, st));
            CU(cudaStreamWaitEvent(P->aux_stream, P->ev_fork, 0));
            if ((s = launch_sat_pull(P, w.S[sc_], Bp, sat_cur, rs, P->aux_stream)) != AFS_OK) return s;
            CU(cudaEventRecord(P->ev_join, P->aux_stream));
        }
        {
            ProfSpan span(P, 1, st);
            launch_var<real, false>(P, a, gx, tiles, rs, st);
        }
        P->last_launches++;
        if (side) CU(cudaStreamWaitEvent(st, P->ev_join, 0));
        bc ^= 1;
        xc = xn;
        { const int tmp = sc_; sc_ = sp_; sp_ = tmp; }   // S[sc_] = words of X_{t+1}, S[sp_] = words of X_t
        pending = true;
        dpending = conv;
        if (retire) {
            // iterate t is merged by the plan; frozen restarts leave with their results; the rest moves to the front
            ProfSpan span(P, 18, st);
            const int xf = (xc + 1) % 3, sf = 3 - sc_ - sp_;
            k_retire_plan<<<1, 1024, 0, st>>>(rs, t, sat_cur, w.best_sat[bc], w.best_step[bc], w.orig[oc], w.moved,
                                              w.best_sat[bc ^ 1], w.best_step[bc ^ 1], w.orig[oc ^ 1], w.rt_src, w.rt_imp,
                                              w.rt_ret, w.rt_ret_sat, w.rt_ret_step, (double)tol, sizeof(real) == 8 ? 1 : 0,
                                              delta + (size_t)(t % 3) * Bp, w.conv[bc], w.conv[bc ^ 1], w.rt_ret_conv);
            k_retire_out<real><<<tg, 256, 0, st>>>(rs, P->n, Bp, XT[xc], w.S[sp_], w.best_bits[bb], w.rt_imp, w.rt_ret,
                                                   w.rt_ret_sat, w.rt_ret_step, w.orig[oc], X, best_assign, best_sat,
                                                   best_step, w.rt_ret_conv, conv_step);
            k_compact<real><<<dim3((P->n + 7) / 8, tiles), 256, 0, st>>>(rs, P->n, Bp, w.rt_src, w.rt_imp, XT[xc], w.S[sp_],
                                                                         w.best_bits[bb], XT[xf], w.S[sf], w.SAT[sf],
                                                                         w.best_bits[bb ^ 1]);
            P->last_launches += 3;
            if (per_restart_masks) {   // the masks move with their restarts
                k_compact_mask<<<dim3((P->n + 7) / 8, tiles), 256, 0, st>>>(rs, P->n, Bp, w.rt_src, maskT[mc], maskT[mc ^ 1]);
                P->last_launches++;
                mc ^= 1;
            }
            bc ^= 1; oc ^= 1; bb ^= 1; xc = xf;
            sp_ = sc_; sc_ = sf;      // the words of X_t are not needed any more: the next pass has nothing to merge
            pending = false;
            dpending = false;
        }
    }
    P->prof.on = false;
    P->long_folded = false;
    // the last iterate: count only, then fold and write out
    const real* Xfin = XT[xc];
    int32_t* sat_fin = w.sat_hist + (size_t)(steps % 3) * Bp;
    if ((s = launch_count<real>(P, Xfin, Bp, sat_fin, rs, st)) != AFS_OK) return s;
    FinArgs<real> f{};
    f.n = P->n; f.B = B; f.Bp = Bp; f.steps = steps; f.XT = Xfin;
    f.sat_prev = pending ? w.sat_hist + (size_t)((steps + 2) % 3) * Bp : nullptr;
    f.sat_fin = sat_fin;
    f.best_sat_in = w.best_sat[bc]; f.best_step_in = w.best_step[bc];
    f.S_prev = w.S[sp_]; f.best_bits = w.best_bits[bb];
    f.X = X; f.best_assign = best_assign; f.best_sat = best_sat; f.best_step = best_step;
    f.rs = rs; f.orig = w.orig[oc];
    f.tol = tol; f.conv_in = w.conv[bc]; f.conv_step = conv_step;
    f.delta_last = dpending ? delta + (size_t)((steps + 2) % 3) * Bp : nullptr;
    k_finalize<real><<<tg, 256, 0, st>>>(f);
    P->last_launches++;
    CU(cudaGetLastError());
    return AFS_OK;
}

// afs_pgd_run_conv: the run, then the Fig. 4-5 outputs of the returned iterate.  The trailing evaluations belong to the
// same call: the launch count and the timing spans of the run survive them.
template <typename real>
static afs_status pgd_run_conv_impl(afs_problem* P, real* X, int32_t B, int32_t max_steps, real lr, const int8_t* mask,
                                    real tol, int8_t* best_assign, int32_t* best_sat, int32_t* best_step,
                                    int32_t* conv_step, int32_t* final_sat, real* final_F, void* stream)
{
    if (!(tol >= real(0)) || !std::isfinite((double)tol)) return AFS_ERR_INVALID_ARG;
    if (P && conv_step && B >= 1) {   // -1 unless the run says otherwise (tol = 0 may take the resident path); on the handle's device
        DeviceScope dev_scope(P);
        if (cudaSetDevice(P->device) != cudaSuccess) { (void)cudaGetLastError(); return AFS_ERR_CUDA; }
        launch_fill_i32(conv_step, (size_t)B, -1, (cudaStream_t)stream);
    }
    afs_status s = pgd_run_impl<real>(P, X, B, max_steps, lr, mask, best_assign, best_sat, best_step, stream, tol, conv_step);
    if (s != AFS_OK) return s;
    int64_t launches = P->last_launches + (conv_step ? 1 : 0);
    const int32_t resident = P->last_resident;
    const std::vector<Profiler::Span> spans = P->prof.spans;
    const size_t used = P->prof.used;
    if (final_sat) { s = round_count_impl<real>(P, X, B, nullptr, final_sat, stream); launches += P->last_launches; }
    if (s == AFS_OK && final_F) { s = eval_grad_impl<real>(P, X, B, final_F, nullptr, stream); launches += P->last_launches; }
    P->last_launches = launches; P->last_resident = resident;
    P->prof.spans = spans; P->prof.used = used;   // the evaluations record no events: the run's spans are intact
    return s;
}

}  // namespace afs
