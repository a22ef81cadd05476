// afs_long_launch.cuh -- launches of the long-constraint kernels (afs_long.cuh), one translation unit per arithmetic
// type (afs_long_f32.cu, afs_long_f64.cu) so that their many instantiations compile beside the rest of the library.
#pragma once
#include "afs_long.cuh"
#include "afs_launch.h"

namespace afs {

template <typename real, int NR, int RPC>
static afs_status launch_long_rpc(afs_problem* P, int bucket, const real* XT, const uint32_t* Sw, const uint32_t* SATw,
                                  int Bp, real* scratch, int32_t* sat, real* fe, cudaStream_t st, int LS, int QS,
                                  size_t smem)
{
    int c0 = P->long_begin[bucket], c1 = P->long_begin[bucket + 1];
    if (smem > 48 * 1024)   // per device and per instantiation: set before every launch, never cached
        CU(cudaFuncSetAttribute(k_long<real, NR, RPC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int ntile = Bp / 32;
    long long blocks = (long long)(c1 - c0) * ntile;
    if (blocks > 0x7fffffffLL) return AFS_ERR_UNSUPPORTED;
    ProfSpan span(P, 8 + NR, st);
    const bool fo = P->long_folded;
    unsigned long long* work = nullptr;
    { afs_status ws = prof_work_slot(P, 8 + NR, st, &work); if (ws != AFS_OK) return ws; }
    k_long<real, NR, RPC><<<(unsigned)blocks, RPC * 32, smem, st>>>(fo ? P->d_long_f : P->d_long, c0,
                                                                    fo ? P->d_long_lits_f : P->d_long_lits,
                                                                    fo ? P->d_long_slots_f : P->d_long_slots, XT, Sw, SATw,
                                                                    ntile, Bp, scratch, (real*)P->ws.bnd, sat, fe, LS, QS,
                                                                    work);
    P->last_launches++;
    return AFS_OK;
}

template <typename real, int NR>
static afs_status launch_long(afs_problem* P, int bucket, const real* XT, const uint32_t* Sw, const uint32_t* SATw, int Bp,
                              real* scratch, int32_t* sat, real* fe, cudaStream_t st)
{
    if (P->long_begin[bucket + 1] <= P->long_begin[bucket]) return AFS_OK;
    int Lmax = P->long_maxL[bucket];
    int LS = ((Lmax + 8 + 31) / 32) * 32;            // list order: L entries + at most 6 neutral ones
    int QS = ((Lmax + 1 + 3 + 3) / 4) * 4 + 4;       // pmf q_0..q_L behind an offset of at most 3
    const size_t per_restart = (size_t)LS * (sizeof(real) + sizeof(uint16_t)) + (size_t)QS * sizeof(real);
    const size_t words = (size_t)LS * 8;             // true + saturated words of the tile
    // warps per CTA (restarts in flight): 8, or 4 where that packs more warps on an SM (the longest rows in fp64)
    const size_t budget = 227 * 1024;
    const int w8 = (int)(budget / (8 * per_restart + words + 1024)) * 8, w4 = (int)(budget / (4 * per_restart + words + 1024)) * 4;
    if (w4 == 0) return AFS_ERR_UNSUPPORTED;
    if (w8 >= w4 || w8 >= 32)
        return launch_long_rpc<real, NR, 8>(P, bucket, XT, Sw, SATw, Bp, scratch, sat, fe, st, LS, QS, 8 * per_restart + words);
    return launch_long_rpc<real, NR, 4>(P, bucket, XT, Sw, SATw, Bp, scratch, sat, fe, st, LS, QS, 4 * per_restart + words);
}

template <typename real>
afs_status launch_long_all(afs_problem* P, const real* XT, const uint32_t* Sw, const uint32_t* SATw, int Bp, real* scratch,
                           int32_t* sat, real* fe, cudaStream_t st)
{
    afs_status s = AFS_OK;
#define LONG_CASE(NRV) if (s == AFS_OK) s = launch_long<real, NRV>(P, NRV - 1, XT, Sw, SATw, Bp, scratch, sat, fe, st);
    LONG_CASE(1) LONG_CASE(2) LONG_CASE(3) LONG_CASE(4) LONG_CASE(5) LONG_CASE(6) LONG_CASE(7) LONG_CASE(8) LONG_CASE(9)
#undef LONG_CASE
    return s;
}

}  // namespace afs
