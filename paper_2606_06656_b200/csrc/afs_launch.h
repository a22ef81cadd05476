// afs_launch.h -- host-side helpers shared by the translation units of libafs_b200 (the library is compiled as several
// objects so that the fp32 product kernels and the fp64 verification build compile in parallel): error macro, the
// per-launch profiler span, and the non-template helpers defined once in afs_common.cu.
#pragma once
#include <algorithm>

#include "afs_internal.h"

#define CU(x)                                \
    do {                                     \
        cudaError_t e_ = (x);                \
        if (e_ != cudaSuccess) {             \
            afs::note_cuda_error(e_, __FILE__, __LINE__); \
            (void)cudaGetLastError();        \
            return AFS_ERR_CUDA;             \
        }                                    \
    } while (0)

namespace afs {

struct RunState;
// the caller's current device is put back when an entry point returns (PyTorch owns device and stream state)
struct DeviceScope {
    int prev = -1;
    explicit DeviceScope(const afs_problem* P) { if (P && cudaGetDevice(&prev) != cudaSuccess) { (void)cudaGetLastError(); prev = -1; } }
    ~DeviceScope() { if (prev >= 0) { cudaSetDevice(prev); (void)cudaGetLastError(); } }
};

void free_workspace(afs_problem* P);
int prof_mark(afs_problem* P, cudaStream_t st);
struct ProfSpan {   // brackets the launches enqueued during its lifetime
    afs_problem* P; cudaStream_t st; int cls, e0;
    ProfSpan(afs_problem* p, int c, cudaStream_t s) : P(p), st(s), cls(c), e0(p->prof.on ? prof_mark(p, s) : -1) {}
    ~ProfSpan() { if (e0 >= 0) { int e1 = prof_mark(P, st); if (e1 >= 0) P->prof.spans.push_back({cls, e0, e1}); } }
};

int fe_pull_grid_x(const afs_problem* P);
inline int fe_pull_parts(const afs_problem* P) { return fe_pull_grid_x(P) * 8; }
afs_status ensure_workspace(afs_problem* P, int Bp, size_t elem, int64_t sat_rows);
afs_status ensure_eval_buffers(afs_problem* P, int Bp, size_t elem);
afs_status enter(afs_problem* P, int32_t B);
afs_status launch_sat_pull(afs_problem* P, const uint32_t* S, int Bp, int32_t* sat, const RunState* rs, cudaStream_t st);
afs_status launch_fill_i32(int32_t* p, size_t n, int32_t v, cudaStream_t st);
afs_status launch_long_fold(afs_problem* P, const int8_t* mask, cudaStream_t st);
afs_status prof_work_slot(afs_problem* P, int cls, cudaStream_t st, unsigned long long** out);

// the long-constraint kernels of one PGD iteration (all length buckets); instantiated in afs_long_f32.cu / _f64.cu
template <typename real>
afs_status launch_long_all(afs_problem* P, const real* XT, const uint32_t* Sw, const uint32_t* SATw, int Bp, real* scratch,
                           int32_t* sat, real* fe, const RunState* rs, cudaStream_t st);

}  // namespace afs
