// afs_long_launch.cuh -- launches of the long-constraint kernels (afs_long.cuh), one translation unit per arithmetic
// type (afs_long_f32.cu, afs_long_f64.cu) so that their instantiations compile beside the rest of the library.
#pragma once
#include "afs_long.cuh"
#include "afs_launch.h"

namespace afs {

template <typename real, int CLS>
static afs_status launch_long_items(afs_problem* P, const LongLists& wl, int set, const real* XT, const uint32_t* Sw,
                                    const uint32_t* SATw, int Bp, real* scratch, real* fe, cudaStream_t st)
{
    constexpr int NR = long_class_rows(CLS);
    constexpr int WPC = sizeof(real) == 8 ? 4 : 8;
    int Lmax = 0;
    for (int i = 0; i < LONG_BUCKETS; ++i) Lmax = std::max(Lmax, P->long_maxL[i]);
    if (CLS > 0 && Lmax <= long_class_maxleff(CLS - 1)) return AFS_OK;   // no constraint can reach this class
    const int LS = 128 * NR, QS = 128 * NR + 8;
    const size_t smem = (size_t)WPC * ((size_t)LS * (sizeof(real) + sizeof(uint16_t)) + (size_t)QS * sizeof(real));
    auto kern = k_long_items<real, NR, WPC>;
    const int ti = sizeof(real) == 8 ? 1 : 0;
    if (smem > 48 * 1024)   // per device and per instantiation: set before every launch, never cached process-wide
        CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (P->long_occ[ti][CLS] == 0) {   // per handle, hence per device
        int occ = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, WPC * 32, smem));
        if (occ < 1) return AFS_ERR_UNSUPPORTED;
        P->long_occ[ti][CLS] = occ;
    }
    // persistent over the work list; never more CTAs than the list can hold entries for
    long long cap = ((long long)P->n_long * Bp + WPC - 1) / WPC;
    const int grid = (int)std::min<long long>((long long)P->sm_count * P->long_occ[ti][CLS], cap < 1 ? 1 : cap);
    ProfSpan span(P, 8 + NR, st);
    const bool fo = P->long_folded;
    unsigned long long* work = nullptr;
    { afs_status ws = prof_work_slot(P, 8 + NR, st, &work); if (ws != AFS_OK) return ws; }
    kern<<<grid, WPC * 32, smem, st>>>(fo ? P->d_long_f : (P->unit_w_mode && P->d_long_u) ? P->d_long_u : P->d_long, fo ? P->d_long_lits_f : P->d_long_lits,
                                        fo ? P->d_long_slots_f : P->d_long_slots, XT, Sw, SATw, Bp / 32, Bp,
                                        scratch + (size_t)P->nslots_a * Bp, (int)P->nslots_a, (int)(P->nslots - P->nslots_a),
                                        (real*)P->ws.bnd, fe, wl.items[CLS], wl.count + set * LONG_CLASSES + CLS, LS, QS,
                                        work, P->d_long_goff, P->ws.long_MI, P->ws.long_MT);
    P->last_launches++;
    return AFS_OK;
}

// classes 4 / 5: one lane per entry (k_long_lane), at most `cap` interior literals
template <typename real>
static afs_status launch_long_lane(afs_problem* P, const LongLists& wl, int set, int cls, int cap, int wpc, int prof_cls,
                                   const real* XT, int Bp, real* scratch, real* fe, cudaStream_t st)
{
    const size_t smem = (size_t)wpc * ((size_t)(3 * cap + 1) * 32 * sizeof(real) + (size_t)cap * 32 * sizeof(uint16_t));
    auto kern = k_long_lane<real>;
    if (smem > 48 * 1024) CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, wpc * 32, smem));
    if (occ < 1) return AFS_ERR_UNSUPPORTED;
    long long cap_blocks = ((long long)P->n_long * Bp + wpc * 32 - 1) / (wpc * 32);
    const int grid = (int)std::min<long long>((long long)P->sm_count * occ, cap_blocks < 1 ? 1 : cap_blocks);
    ProfSpan span(P, prof_cls, st);
    const bool fo = P->long_folded;
    unsigned long long* work = nullptr;
    { afs_status ws = prof_work_slot(P, prof_cls, st, &work); if (ws != AFS_OK) return ws; }
    kern<<<grid, wpc * 32, smem, st>>>(fo ? P->d_long_f : (P->unit_w_mode && P->d_long_u) ? P->d_long_u : P->d_long, fo ? P->d_long_lits_f : P->d_long_lits,
                                       fo ? P->d_long_slots_f : P->d_long_slots, XT, Bp, scratch + (size_t)P->nslots_a * Bp,
                                       (int)P->nslots_a, (int)(P->nslots - P->nslots_a), (real*)P->ws.bnd, fe, wl.items[cls],
                                       wl.count + set * LONG_CLASSES + cls, cap, P->d_long_goff, P->ws.long_MI, P->ws.long_MT, work);
    P->last_launches++;
    return AFS_OK;
}

template <typename real>
afs_status launch_long_all(afs_problem* P, const real* XT, const uint32_t* Sw, const uint32_t* SATw, int Bp, real* scratch,
                           int32_t* sat, real* fe, const RunState* rs, cudaStream_t st)
{
    if (P->n_long == 0) return AFS_OK;
    // k_glong addresses the pair table and the class's rows with 32-bit element offsets
    if ((unsigned long long)P->n_long * (unsigned long long)Bp * 2ull >= (1ull << 32) ||
        (unsigned long long)(P->nslots - P->nslots_a) * 32ull >= (1ull << 32)) return AFS_ERR_UNSUPPORTED;
    LongLists wl;
    for (int k = 0; k < LONG_CLASSES; ++k) wl.items[k] = P->ws.long_items[k];
    wl.count = P->ws.long_count;
    const int set = (int)(P->long_iter++ & 1);
    const bool fo = P->long_folded;
    const int ntile = Bp / 32;
    const long long warps = (long long)P->n_long * ntile;
    if ((warps + 3) / 4 > 0x7fffffffLL) return AFS_ERR_UNSUPPORTED;
    {
        ProfSpan span(P, 5, st);
        // persistent over the (constraint, active tile) pairs: one resident wave of CTAs
        k_long_scan<real><<<(unsigned)std::min<long long>((warps + 3) / 4, (long long)P->sm_count * 16), 128, 0, st>>>(fo ? P->d_long_f : (P->unit_w_mode && P->d_long_u) ? P->d_long_u : P->d_long, (int)P->n_long,
                                                                      fo ? P->d_long_lits_f : P->d_long_lits, Sw, SATw, ntile,
                                                                      Bp, (real*)P->ws.bnd, sat, fe, wl, set, rs, P->d_long_goff, P->ws.long_MI,
                                                                      P->ws.long_MT);
        P->last_launches++;
    }
    afs_status s = launch_long_items<real, 0>(P, wl, set, XT, Sw, SATw, Bp, scratch, fe, st);
    if (s == AFS_OK) s = launch_long_items<real, 1>(P, wl, set, XT, Sw, SATw, Bp, scratch, fe, st);
    if (s == AFS_OK) s = launch_long_items<real, 2>(P, wl, set, XT, Sw, SATw, Bp, scratch, fe, st);
    if (s == AFS_OK) s = launch_long_items<real, 3>(P, wl, set, XT, Sw, SATw, Bp, scratch, fe, st);
    if (s == AFS_OK) s = launch_long_lane<real>(P, wl, set, 4, long_lane_cap(4), 8, 10, XT, Bp, scratch, fe, st);
    if (s == AFS_OK) s = launch_long_lane<real>(P, wl, set, 5, long_lane_cap(5), 8, 14, XT, Bp, scratch, fe, st);
    if (s == AFS_OK) s = launch_long_lane<real>(P, wl, set, 6, long_lane_cap(6), 4, 12, XT, Bp, scratch, fe, st);
    return s;
}

}  // namespace afs
