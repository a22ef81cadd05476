// afs_common.cu -- the parts of libafs_b200 that do not depend on the arithmetic type: workspace management, the
// per-launch profiler, the integer / bit-word kernels' launches, and the host-buffer entry point.
#include <algorithm>
#include <cmath>
#include <cstdio>

#include "afs_kernels.cuh"
#include "afs_launch.h"
#include "afs_retire.cuh"

using namespace afs;

namespace afs {

__global__ void k_fill_i32(int32_t* p, size_t n, int32_t v)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

// Folding of the run's fixed variables (G16), once per afs_pgd_run with a mask: a literal of a fixed
// variable is a constant of the run -- true or false for every restart and every iteration -- so it leaves the list,
// a fixed true one lowers k by one, and the gradient row of its slot is never read (a fixed variable does not move).
// warp = constraint; the compacted lists keep the constraint's offset.  EK / CARD only (the LONG class).
__global__ void __launch_bounds__(128) k_long_fold(const LongCon* __restrict__ cons, const uint32_t* __restrict__ lits,
                                                   const int32_t* __restrict__ slots, int n_long,
                                                   const int8_t* __restrict__ mask, LongCon* __restrict__ cons_f,
                                                   uint32_t* __restrict__ lits_f, int32_t* __restrict__ slots_f)
{
    const int lane = threadIdx.x & 31;
    const int c = blockIdx.x * 4 + (threadIdx.x >> 5);
    if (c >= n_long) return;
    LongCon lc = cons[c];
    const unsigned lt = (1u << lane) - 1u;
    int out = 0, ftrue = 0;
    for (int j0 = 0; j0 < lc.L; j0 += 32) {
        const int j = j0 + lane;
        const bool act = j < lc.L;
        const uint32_t w = act ? lits[lc.off + j] : 0u;
        const int mk = act ? (int)mask[w & LIT_VAR] : 0;
        const bool fixed = act && mk != 0;
        const bool keep = act && !fixed;
        ftrue += __popc(__ballot_sync(0xffffffffu, fixed && ((mk < 0) != ((w >> 31) != 0))));   // True is -1
        const unsigned m = __ballot_sync(0xffffffffu, keep);
        if (keep) {
            const int pos = out + __popc(m & lt);
            lits_f[lc.off + pos] = w;
            slots_f[lc.off + pos] = slots[lc.off + j];
        }
        out += __popc(m);
    }
    if (lane == 0) {
        lc.L = out;
        lc.k -= ftrue;
        lc.tA = lc.tB = 0;
        lc.wA = lc.wB = 0.f;
        // d_t of P:L52 on the folded constraint: CARD >= k: +1 at k-1;  EK: +1 at k-1, -1 at k (indices 0..L-1 only)
        if (lc.k - 1 >= 0 && lc.k - 1 <= out - 1) { lc.tA = lc.k - 1; lc.wA = 1.f; }
        if (lc.type == AFS_EK && lc.k >= 0 && lc.k <= out - 1) { lc.tB = lc.k; lc.wB = -1.f; }
        cons_f[c] = lc;
    }
}


static void free_ptr(void*& p) { if (p) cudaFree(p); p = nullptr; }
template <typename T> static void free_ptr(T*& p) { if (p) cudaFree(p); p = nullptr; }

void free_workspace(afs_problem* P)
{
    Workspace& w = P->ws;
    free_ptr(w.XT[0]); free_ptr(w.XT[1]); free_ptr(w.XT[2]); free_ptr(w.scratch); free_ptr(w.aux[0]); free_ptr(w.aux[1]);
    free_ptr(w.sat_hist); free_ptr(w.best_sat[0]); free_ptr(w.best_sat[1]);
    free_ptr(w.best_step[0]); free_ptr(w.best_step[1]); free_ptr(w.S[0]); free_ptr(w.S[1]); free_ptr(w.S[2]); free_ptr(w.SAT[0]); free_ptr(w.SAT[1]); free_ptr(w.SAT[2]);
    free_ptr(w.bnd); free_ptr(w.GL); free_ptr(w.best_bits[1]); free_ptr(w.orig[0]); free_ptr(w.orig[1]); free_ptr(w.moved);
    free_ptr(w.rs); free_ptr(w.rt_src); free_ptr(w.rt_imp); free_ptr(w.rt_ret); free_ptr(w.rt_ret_sat); free_ptr(w.rt_ret_step); free_ptr(w.rt_ret_conv); free_ptr(w.maskT); free_ptr(w.gm_part); free_ptr(w.conv[0]); free_ptr(w.conv[1]); free_ptr(w.delta);
    for (int k = 0; k < 7; ++k) free_ptr(w.long_items[k]);
    free_ptr(w.long_count); free_ptr(w.long_MI); free_ptr(w.long_MT); free_ptr(w.best_bits[0]);
    free_ptr(w.fe_med); free_ptr(w.fe_long); free_ptr(w.fe_cm); free_ptr(w.f_part);
    free_ptr(w.mask_dev); free_ptr(w.host_stage_X); free_ptr(w.host_stage_assign);
    free_ptr(w.host_stage_sat); free_ptr(w.host_stage_step);
    w = Workspace();
}


// ---- per-launch timing (afs_profile_read) -------------------------------------------------------------------------
int prof_mark(afs_problem* P, cudaStream_t st)
{
    Profiler& pr = P->prof;
    if (pr.used == pr.pool.size()) {
        cudaEvent_t e;
        if (cudaEventCreate(&e) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
        pr.pool.push_back(e);
    }
    if (cudaEventRecord(pr.pool[pr.used], st) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
    return (int)pr.used++;
}

int fe_pull_grid_x(const afs_problem* P) { int g = (int)((P->n_pull + 63) / 64); return g < 1 ? 1 : (g > 2048 ? 2048 : g); }

template <typename T>
static afs_status dev_alloc(T** p, size_t count, size_t& total)
{
    size_t bytes = (count ? count : 1) * sizeof(T);
    if (cudaMalloc((void**)p, bytes) != cudaSuccess) { (void)cudaGetLastError(); *p = nullptr; return AFS_ERR_ALLOC; }
    total += bytes;
    return AFS_OK;
}

// (re)allocate the core workspace for padded batch Bp, element size `elem`, and `sat_rows` count rows
afs_status ensure_workspace(afs_problem* P, int Bp, size_t elem, int64_t sat_rows)
{
    Workspace& w = P->ws;
    if (w.Bp >= Bp && w.elem >= elem && w.sat_rows >= sat_rows) return AFS_OK;
    int nBp = Bp > w.Bp ? Bp : w.Bp;
    size_t nelem = elem > w.elem ? elem : w.elem;
    int64_t nrows = sat_rows > w.sat_rows ? sat_rows : w.sat_rows;
    CU(cudaDeviceSynchronize());
    afs::free_workspace(P);
    size_t tot = 0;
    afs_status st = AFS_OK;
    auto A = [&](auto** p, size_t cnt) { if (st == AFS_OK) st = dev_alloc(p, cnt, tot); };
    const size_t n = (size_t)P->n, ntile = (size_t)nBp / 32;
    A((unsigned char**)&w.XT[0], n * nBp * nelem);
    A((unsigned char**)&w.XT[1], n * nBp * nelem);
    A((unsigned char**)&w.XT[2], n * nBp * nelem);
    A((unsigned char**)&w.scratch, (size_t)P->nslots * nBp * nelem);
    A((unsigned char**)&w.aux[0], (size_t)P->med_nnz * nBp * nelem);
    A((unsigned char**)&w.aux[1], (size_t)(P->med_two ? P->med_nnz : 0) * nBp * nelem);
    A(&w.sat_hist, (size_t)nrows * nBp);
    A(&w.best_sat[0], (size_t)nBp); A(&w.best_sat[1], (size_t)nBp);
    A(&w.best_step[0], (size_t)nBp); A(&w.best_step[1], (size_t)nBp);
    A(&w.S[0], n * ntile); A(&w.S[1], n * ntile); A(&w.S[2], n * ntile);
    A(&w.best_bits[0], n * ntile); A(&w.best_bits[1], n * ntile);
    A(&w.SAT[0], n * ntile); A(&w.SAT[1], n * ntile); A(&w.SAT[2], n * ntile);
    A(&w.orig[0], (size_t)nBp); A(&w.orig[1], (size_t)nBp); A(&w.moved, (size_t)nBp);
    A(&w.rs, (size_t)1); A(&w.rt_src, (size_t)nBp); A(&w.rt_imp, (size_t)nBp); A(&w.rt_ret, (size_t)nBp);
    A(&w.rt_ret_sat, (size_t)nBp); A(&w.rt_ret_step, (size_t)nBp); A(&w.rt_ret_conv, (size_t)nBp);
    A(&w.conv[0], (size_t)nBp); A(&w.conv[1], (size_t)nBp); A((unsigned long long**)&w.delta, (size_t)3 * nBp);
    A((unsigned char**)&w.bnd, (size_t)P->n_long * nBp * 2 * nelem);
    A((unsigned char**)&w.GL, (P->n_long > 0 ? n : 0) * nBp * nelem);
    for (int k = 0; k < 7; ++k) A(&w.long_items[k], (size_t)P->n_long * nBp);
    A(&w.long_count, (size_t)16);
    A(&w.long_MI, (size_t)P->long_grows * nBp); A(&w.long_MT, (size_t)P->long_grows * nBp);
    if (st != AFS_OK) { afs::free_workspace(P); return st; }
    CU(cudaMemset(w.long_count, 0, 16 * sizeof(int)));
    w.Bp = nBp; w.elem = nelem; w.sat_rows = nrows; w.bytes = tot;
    return AFS_OK;
}

afs_status ensure_eval_buffers(afs_problem* P, int Bp, size_t elem)
{
    Workspace& w = P->ws;
    if (w.fe_Bp >= Bp && w.fe_med) return AFS_OK;
    CU(cudaDeviceSynchronize());
    free_ptr(w.fe_med); free_ptr(w.fe_long); free_ptr(w.fe_cm); free_ptr(w.f_part);
    size_t tot = 0;
    afs_status st = AFS_OK;
    auto A = [&](auto** p, size_t cnt) { if (st == AFS_OK) st = dev_alloc(p, cnt, tot); };
    size_t e = w.elem > elem ? w.elem : elem;
    A((unsigned char**)&w.fe_med, (size_t)P->n_med * w.Bp * e);
    A((unsigned char**)&w.fe_long, (size_t)P->n_long * w.Bp * e);
    A((unsigned char**)&w.fe_cm, (size_t)P->n_cm * w.Bp * e);
    A((unsigned char**)&w.f_part, (size_t)fe_pull_parts(P) * w.Bp * e);
    if (st != AFS_OK) return st;
    w.fe_Bp = w.Bp; w.bytes += tot;
    return AFS_OK;
}

// S9 of the PULL class from the sign words of the iterate (bit-parallel over restarts)
afs_status launch_sat_pull(afs_problem* P, const uint32_t* S, int Bp, int32_t* sat, const RunState* rs, cudaStream_t st)
{
    if (P->n_pull == 0) return AFS_OK;
    const int ntile = Bp / 32;
    const int tpt = ntile % 4 == 0 ? 4 : ntile % 2 == 0 ? 2 : 1;
    const int gy = ntile / tpt;
    const int m = (int)P->n_pull;
    int gx = (m + 255) / 256;                               // 8 warps x 32 clauses per CTA and pass
    const int cap = (P->sm_count * 8 + gy - 1) / gy;        // enough CTAs to fill the chip, grid-stride beyond
    if (gx > cap) gx = cap < 1 ? 1 : cap;
    dim3 grid(gx, gy);
    ProfSpan span(P, 2, st);
    if (tpt == 4) k_sat_pull<4><<<grid, 256, 0, st>>>(P->d_pcp, m, S, ntile, sat, rs);
    else if (tpt == 2) k_sat_pull<2><<<grid, 256, 0, st>>>(P->d_pcp, m, S, ntile, sat, rs);
    else k_sat_pull<1><<<grid, 256, 0, st>>>(P->d_pcp, m, S, ntile, sat, rs);
    P->last_launches++;
    return AFS_OK;
}

afs_status enter(afs_problem* P, int32_t B)
{
    if (!P || B < 1) return AFS_ERR_INVALID_ARG;
    // row offsets inside the kernels are 32-bit byte offsets: n * Bp * 8 must stay below 4 GiB
    if ((unsigned long long)P->n * (unsigned long long)(((B + 31) / 32) * 32) * 8ull >= (1ull << 32)) return AFS_ERR_UNSUPPORTED;
    if (cudaSetDevice(P->device) != cudaSuccess) { (void)cudaGetLastError(); return AFS_ERR_CUDA; }
    P->last_launches = 0;
    P->long_folded = false;
    P->prof.on = false;
    P->prof.spans.clear();
    P->prof.used = 0;
    return AFS_OK;
}

afs_status launch_fill_i32(int32_t* p, size_t n, int32_t v, cudaStream_t st)
{
    k_fill_i32<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(p, n, v);
    return AFS_OK;
}

// the fixed variables' literals leave the long constraints for this run (k_long_fold)
afs_status launch_long_fold(afs_problem* P, const int8_t* mask, cudaStream_t st)
{
    k_long_fold<<<(unsigned)((P->n_long + 3) / 4), 128, 0, st>>>(P->d_long, P->d_long_lits, P->d_long_slots, (int)P->n_long,
                                                               mask, P->d_long_f, P->d_long_lits_f, P->d_long_slots_f);
    P->last_launches++;
    P->long_folded = true;
    return AFS_OK;
}

// timing mode: the counter block of kernel class `cls` (allocated on first use)
afs_status prof_work_slot(afs_problem* P, int cls, cudaStream_t st, unsigned long long** out)
{
    *out = nullptr;
    if (!P->prof.on) return AFS_OK;
    if (!P->prof.d_work) {
        CU(cudaMalloc((void**)&P->prof.d_work, sizeof(unsigned long long) * PROF_CLASSES * 32));
        CU(cudaMemsetAsync(P->prof.d_work, 0, sizeof(unsigned long long) * PROF_CLASSES * 32, st));
    }
    *out = P->prof.d_work + cls * 32;
    return AFS_OK;
}

}  // namespace afs

extern "C" afs_status afs_profile_read(afs_problem* P, double* ms, int64_t* launches, int32_t n)
{
    DeviceScope dev_scope(P);
    if (P && cudaSetDevice(P->device) != cudaSuccess) { (void)cudaGetLastError(); return AFS_ERR_CUDA; }
    if (!P || !ms || !launches || n < 0 || n > PROF_CLASSES) return AFS_ERR_INVALID_ARG;
    Profiler& pr = P->prof;
    if (pr.used > 0) CU(cudaEventSynchronize(pr.pool[pr.used - 1]));
    // spans of the pull-clause counts are recorded on the library's second stream, which the caller's stream joins
    // only AFTER its own last event: wait for that stream too before reading their events
    if (pr.used > 0 && P->aux_stream) CU(cudaStreamSynchronize(P->aux_stream));
    for (const Profiler::Span& sp : pr.spans) {
        float t = 0.f;
        CU(cudaEventElapsedTime(&t, pr.pool[sp.e0], pr.pool[sp.e1]));
        if (sp.cls < n) { ms[sp.cls] += (double)t; launches[sp.cls] += 1; }
    }
    pr.spans.clear();
    pr.used = 0;
    if (pr.d_work) {
        unsigned long long h[PROF_CLASSES * 32];
        CU(cudaMemcpy(h, pr.d_work, sizeof(h), cudaMemcpyDeviceToHost));
        CU(cudaMemset(pr.d_work, 0, sizeof(h)));
        for (int c = 0; c < PROF_CLASSES; ++c)
            for (int i = 0; i < 32; ++i) pr.work[c] += (double)h[c * 32 + i];
    }
    return AFS_OK;
}

extern "C" afs_status afs_profile_flops(afs_problem* P, double* flops, int32_t n)
{
    if (!P || !flops || n < 0 || n > PROF_CLASSES) return AFS_ERR_INVALID_ARG;
    for (int c = 0; c < n; ++c) { flops[c] += P->prof.work[c]; }
    for (int c = 0; c < PROF_CLASSES; ++c) P->prof.work[c] = 0.0;
    return AFS_OK;
}

extern "C" afs_status afs_pgd_run_host(afs_problem* P, float* X, int32_t B, int32_t steps, float lr, const int8_t* mask,
                                       int8_t* best_assign, int32_t* best_sat, int32_t* best_step, void* stream)
{
    DeviceScope dev_scope(P);
    afs_status s = enter(P, B);
    if (s != AFS_OK) return s;
    if (!X) return AFS_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    Workspace& w = P->ws;
    const size_t n = (size_t)P->n;
    // the core workspace first: growing it later would free these staging buffers
    if ((s = ensure_workspace(P, ((B + 31) / 32) * 32, sizeof(float), 3)) != AFS_OK) return s;
    if (w.host_stage_B < B) {
        CU(cudaDeviceSynchronize());
        free_ptr(w.mask_dev); free_ptr(w.host_stage_X); free_ptr(w.host_stage_assign);
        free_ptr(w.host_stage_sat); free_ptr(w.host_stage_step);
        size_t tot = 0;
        afs_status a = AFS_OK;
        auto A = [&](auto** p, size_t cnt) { if (a == AFS_OK) a = dev_alloc(p, cnt, tot); };
        A(&w.mask_dev, n);
        A((float**)&w.host_stage_X, n * B);
        A(&w.host_stage_assign, n * B);
        A(&w.host_stage_sat, (size_t)B);
        A(&w.host_stage_step, (size_t)B);
        if (a != AFS_OK) return a;
        w.host_stage_B = B; w.bytes += tot;
    }
    float* dX = (float*)w.host_stage_X;
    CU(cudaMemcpyAsync(dX, X, n * B * sizeof(float), cudaMemcpyHostToDevice, st));
    if (mask) CU(cudaMemcpyAsync(w.mask_dev, mask, n, cudaMemcpyHostToDevice, st));
    s = afs_pgd_run(P, dX, B, steps, lr, mask ? w.mask_dev : nullptr, w.host_stage_assign, w.host_stage_sat,
                    w.host_stage_step, stream);
    if (s != AFS_OK) return s;
    CU(cudaMemcpyAsync(X, dX, n * B * sizeof(float), cudaMemcpyDeviceToHost, st));
    if (best_assign) CU(cudaMemcpyAsync(best_assign, w.host_stage_assign, n * B, cudaMemcpyDeviceToHost, st));
    if (best_sat) CU(cudaMemcpyAsync(best_sat, w.host_stage_sat, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    if (best_step) CU(cudaMemcpyAsync(best_step, w.host_stage_step, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    return AFS_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// afs_fp32_fma_peak: the plain-FP32 ceiling of this GPU, measured ("measure an FMA micro-benchmark on
// the box").  Not on the product path: bench.py calls it for the denominator of the "alu" roofline.  Every thread runs
// 8 independent FFMA chains; 2 CTAs x 1024 threads per SM keep all four schedulers of every SM issuing.
// ---------------------------------------------------------------------------------------------------------------------
namespace afs {
__global__ void __launch_bounds__(1024, 2) k_fma_peak(float* __restrict__ out, int iters, float a, float b)
{
    float x[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) x[i] = (float)(threadIdx.x + i) * 1e-3f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 8; ++r)
#pragma unroll
            for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += x[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}
}  // namespace afs

extern "C" afs_status afs_fp32_fma_peak(int32_t device, double* tflops)
{
    if (!tflops) return AFS_ERR_INVALID_ARG;
    *tflops = 0.0;
    int ndev = 0, prev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) { (void)cudaGetLastError(); return AFS_ERR_CUDA; }
    CU(cudaGetDevice(&prev));
    CU(cudaSetDevice(device));
    cudaDeviceProp prop;
    CU(cudaGetDeviceProperties(&prop, device));
    const int grid = prop.multiProcessorCount * 2, iters = 4096;
    float* out = nullptr;
    CU(cudaMalloc((void**)&out, (size_t)grid * 1024 * sizeof(float)));
    cudaEvent_t e0, e1;
    CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 6; ++rep) {   // the first repetition is the warm-up
        CU(cudaEventRecord(e0, 0));
        k_fma_peak<<<grid, 1024>>>(out, iters, 0.999f, 1e-3f);
        CU(cudaEventRecord(e1, 0));
        CU(cudaEventSynchronize(e1));
        float ms = 0.f;
        CU(cudaEventElapsedTime(&ms, e0, e1));
        const double fl = (double)grid * 1024.0 * iters * 64.0 * 2.0;
        if (rep > 0 && ms > 0.f) best = std::max(best, fl / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    cudaSetDevice(prev);
    *tflops = best;
    return AFS_OK;
}
