// afs_internal.h -- host-side problem representation shared by the translation units of libafs_b200.
// Not part of the ABI (include/afs.h is).  No code from oracle/ is used here or anywhere in csrc/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/afs.h"

namespace afs {

struct RunState;

// ---- literal word: bit 31 = negated literal, bits 0..30 = variable index -------------------------------------
constexpr uint32_t LIT_NEG = 0x80000000u;
constexpr uint32_t LIT_VAR = 0x7fffffffu;

// ---- execution classes (decided at create; S0 of the path) ---------------------------------------------------
//  PULL : OR / XOR / NAE with L <= PULL_MAX_LEN.  No gradient is materialised: the variable pass recomputes each
//         occurrence's leave-one-out product from the other literals (deterministic by construction).
//  MED  : thread per (constraint, restart): OR / XOR beyond the pull lengths and NAE / EO / AMO of any length;
//         prefix states stored per literal in private rows (aux), suffix carried backwards in registers.
//  CMED : EK / CARD with L <= 64: thread per (constraint, restart), the pmf in the warp's shared-memory buffer.
//  LONG : warp per (constraint, restart), count-basis DP + stable-direction leave-one-out recurrences:
//         EK/CARD longer than 64.
constexpr int PULL_MAX_LEN = 5;
constexpr int LONG_MAX_LEN = 1144;   // = long_class_maxleff(3): the item kernel's lists of 9 x 128 entries hold Leff + 6 <= 1150 padded entries
constexpr int LONG_BUCKETS = 9;      // NR = 1..9 rows of 128 pmf cells

// pull streams (S0 output for the PULL class).  Per variable its occurrences are grouped into RUNS of equal
// (kind, number of other literals); a run is `count` occurrences x `nother` entries, one uint32 per OTHER literal:
//   entry       bits 0..23 variable | 30 occurrence sign (first entry of the occurrence only) | 31 literal negated
//   occurrence sign = own literal negated XOR (XOR constraint with even parity): the leave-one-out product enters
//               the variable's gradient with that sign
//   run word    bits 30..31 kind | 27..29 nother (1..4) | 0..26 count
// Unit clauses (no other literal) contribute a constant to the gradient: pull_gconst[v].
constexpr uint32_t PE_VAR = 0x00ffffffu, PE_SIGN = 1u << 30, PE_NEG = 1u << 31;
constexpr uint32_t PH_KIND_OR = 0, PH_KIND_XOR = 1, PH_KIND_NAE = 2;
constexpr int MAX_VARS = 1 << 24;
constexpr int CM_BUCKETS = 4;        // EK / CARD with L <= 64, ordered by length class 16, 32, 48, 64
constexpr int CM_MAX_LEN = 64;

struct MedCon {        // 20 bytes
    int32_t off;       // first literal in med_lits / med_slots
    int32_t L;
    int32_t type;
    int32_t k;
    float w;           // weight w_k of the constraint in eq. (5) (1 unless created with weights)
};

struct LongCon {       // 36 bytes
    int32_t off;       // first literal in long_lits / long_slots
    int32_t L;
    int32_t type;
    int32_t k;
    int32_t tA, tB;    // leave-one-out pmf indices entering the gradient (true-count index, 0..L-1)
    float wA, wB;      // their weights d_t in {-1, 0, +1}
    float w;           // weight w_k of the constraint in eq. (5)
};

struct PullClause {    // one PULL-class clause packed for the bit-parallel count: header + its <= 5 literal words, 32 bytes
    uint32_t hdr;      // bits 0..2 L | 3..4 kind (PH_KIND_*) | 5 XOR parity k
    uint32_t lit[PULL_MAX_LEN];
    uint32_t pad[2];
};

struct CountCon {      // generic forward CSR entry for the count-only kernel: 16 bytes
    int64_t off;
    int32_t L;
    int16_t type;
    int16_t pad;
    int32_t k;
    int32_t pad2;
};

// ---- tile-resident kernel (afs_resident.cuh): static split of one tile's work over the C CTAs of a cluster ----------
struct ResItem {       // one MED-class constraint: idx into d_med (code unused)
    uint32_t code;
    uint32_t idx;
};
constexpr int RES_PLANS = 8;   // cluster sizes 1 .. 8 (plan i: i + 1 CTAs per tile)
struct ResPlan {
    int C = 0;
    int32_t* d_var_begin = nullptr;    // [C+1] contiguous variable ranges, balanced by pull + reduction work
    int32_t* d_item_begin = nullptr;   // [C+1] ranges of d_items, each rank's items heaviest first
    ResItem* d_items = nullptr;
    int32_t* d_cm_begin = nullptr;     // [C+1] ranges of d_cm_items
    int32_t* d_cm_items = nullptr;     // CMED constraints (indices into d_cm), each rank's heaviest first
    int32_t* d_pc_begin = nullptr;     // [C+1] ranges of the pull clauses whose counts the rank takes
    // capacities (max over ranks) of the index streams a CTA may stage in shared memory
    int cap_words = 0, cap_runs = 0, cap_own = 0, cap_plits = 0, cap_cm = 0, cap_push = 0;
};

// ---- per-launch device timing (afs_set_option 1, afs_profile_read): CUDA events on the caller's stream around the
// launches of every `stride`-th PGD iteration, summed per kernel class (afs_kernel_class in afs.h)
constexpr int PROF_CLASSES = 19;
struct Profiler {
    int stride = 0;                       // 0 = off
    bool on = false;                      // the iteration being enqueued is sampled
    std::vector<cudaEvent_t> pool;
    size_t used = 0;
    struct Span { int cls, e0, e1; };
    std::vector<Span> spans;
    unsigned long long* d_work = nullptr;   // [PROF_CLASSES][32] state-dependent algorithmic flops counted by the kernels
    double work[PROF_CLASSES] = {0};        // of the timed launches (k_long only), summed at afs_profile_read
};

// records cudaGetErrorString(e) + location for afs_last_error_message()
void note_cuda_error(cudaError_t e, const char* file, int line);

struct Workspace {
    // all sized for (Bp, steps) below; grown on demand
    int32_t Bp = 0;
    int64_t sat_rows = 0;
    void* XT[3] = {nullptr, nullptr, nullptr};   // real [n][Bp]: X_t, X_{t+1} and the target of a compaction, in rotation
    void* scratch = nullptr;               // real [nslots][Bp]
    void* aux[2] = {nullptr, nullptr};     // real [med_nnz][Bp] prefix states of the MED class
    int32_t* sat_hist = nullptr;           // [sat_rows][Bp]
    int32_t* best_sat[2] = {nullptr, nullptr};
    int32_t* best_step[2] = {nullptr, nullptr};
    uint32_t* S[3] = {nullptr, nullptr, nullptr};   // sign bits [n][Bp/32]: bit r of word (v, tile) = "x_v < 0" for restart 32 tile + r
    uint32_t* SAT[3] = {nullptr, nullptr, nullptr}; // saturation bits, same layout: |x_v| = 1 (on the boundary of the cube)
    void* GL = nullptr;                    // real [n][Bp]: the LONG class's share of the gradient (k_glong -> k_var)
    void* bnd = nullptr;                   // real [n_long][Bp][2]: dFE/dy of a boundary literal at y = +1 / y = -1
    uint4* long_items[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // work lists of the long-constraint kernels, by size class
    uint32_t* long_MI = nullptr;           // [long_grows][Bp] per group of 32 literals and restart: interior-literal mask,
    uint32_t* long_MT = nullptr;           //                  literal-true mask (k_long_scan -> k_long_items)
    int* long_count = nullptr;             // [2][7] their lengths, two sets used alternately
    uint32_t* best_bits[2] = {nullptr, nullptr};   // [n][Bp/32]
    // retirement of restarts at a fixed point (afs_retire.cuh)
    afs::RunState* rs = nullptr;
    int32_t* orig[2] = {nullptr, nullptr}; // [Bp] caller's restart index of every working column, -1 = none
    int32_t* moved = nullptr;              // [Bp] the column changed in the step a retirement follows
    int32_t* rt_src = nullptr;             // [Bp] plan: old column of every new one
    uint8_t* rt_imp = nullptr;             // [Bp] plan: the pending iterate improved the column's best
    int32_t* rt_ret = nullptr;             // [Bp] plan: frozen columns, with their final best record
    int32_t* rt_ret_sat = nullptr;
    int32_t* rt_ret_step = nullptr;
    int32_t* rt_ret_conv = nullptr;
    // convergence detection (afs_pgd_run_conv)
    int8_t* maskT = nullptr;               // [n][Bp] per-restart masks, transposed (afs_pgd_run_masks); allocated on first use
    int64_t maskT_elems = 0;
    int32_t* conv[2] = {nullptr, nullptr}; // [Bp] steps after which the column stopped, -1 = running
    void* delta = nullptr;                 // [3][Bp] 8-byte cells: max |dX| of a step as order-preserving integer bits
    void* fe_med = nullptr;                // real [n_med][Bp]      (eval_grad only)
    void* fe_long = nullptr;               // real [n_long][Bp]
    void* fe_cm = nullptr;                 // real [n_cm][Bp]
    void* f_part = nullptr;                // real [n_parts][Bp]
    void* gm_part = nullptr;               // real [m][Bp/32] per-constraint gradient magnitude, one partial per restart tile
    int64_t gm_elems = 0;
    int32_t fe_Bp = 0;
    int8_t* mask_dev = nullptr;            // staging for afs_pgd_run_host
    void* host_stage_X = nullptr;          // device X[B,n] staging for afs_pgd_run_host
    int8_t* host_stage_assign = nullptr;
    int32_t* host_stage_sat = nullptr;
    int32_t* host_stage_step = nullptr;
    int64_t host_stage_B = 0;
    size_t elem = 0;                       // sizeof(real) the buffers were sized for
    size_t bytes = 0;
};

}  // namespace afs

struct afs_problem {
    int32_t n = 0, m = 0;
    int64_t nnz = 0;
    int device = 0;
    int sm_count = 148;

    // ---- device tables -------------------------------------------------------------------------------------
    int32_t* d_pull_ptr = nullptr;      // [n+1] entry offsets of each variable's pull stream
    uint32_t* d_pull_words = nullptr;   // entries
    int64_t pull_words = 0;
    int32_t* d_run_ptr = nullptr;       // [n+1] offsets into d_runs
    uint32_t* d_runs = nullptr;         // run descriptors
    float* d_pull_gconst = nullptr;     // [n] constant gradient of unit clauses
    afs::CountCon* d_pc = nullptr;      // the PULL constraints alone (forward CSR), for counts and objective
    uint32_t* d_pc_lits = nullptr;
    afs::PullClause* d_pcp = nullptr;   // the same clauses packed for the bit-parallel counts
    int32_t* d_slot_ptr = nullptr;      // [n+1] scratch rows of each variable (transposed-CSR order)
    int32_t* d_lslot_ptr = nullptr;     // [n+1] rows of the LONG class of each variable, relative to row nslots_a
    int32_t* d_lslot_info = nullptr;    // per LONG-class row: (index in d_long) << 1 | literal negated
    int64_t nslots = 0;                 // all scratch rows: [0, nslots_a) MED / CMED literals, [nslots_a, nslots) LONG literals
    int64_t nslots_a = 0;

    afs::MedCon* d_med = nullptr;       // sorted by bucket
    uint32_t* d_med_lits = nullptr;
    int32_t* d_med_slots = nullptr;
    int64_t med_nnz = 0;                // literals of the MED class = rows of the aux buffers
    bool med_two = false;               // some MED constraint carries a two-component prefix state (NAE / EO / AMO)

    afs::LongCon* d_long = nullptr;     // sorted by bucket (NR), longest first inside a bucket
    uint32_t* d_long_lits = nullptr;
    int32_t* d_long_slots = nullptr;
    // the same class with the literals of the run's fixed variables folded away (k_long_fold, once per afs_pgd_run with
    // a mask): compacted literal / slot lists at the same offsets, L and k reduced, targets recomputed
    afs::LongCon* d_long_f = nullptr;
    uint32_t* d_long_lits_f = nullptr;
    int32_t* d_long_slots_f = nullptr;
    int32_t* d_long_goff = nullptr;     // [n_long] first mask row of each constraint (rows = groups of 32 literals)
    int64_t long_grows = 0;             // mask rows in all
    int64_t long_nnz = 0;
    bool long_folded = false;           // the launches of the current call use the folded lists
    uint64_t long_iter = 0;             // launches of the long-constraint pass so far (parity selects the counter set)
    int long_occ[2][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}};   // resident CTAs per SM of the item kernels (per type, size class)
    int32_t long_begin[afs::LONG_BUCKETS + 1] = {0};
    int32_t long_maxL[afs::LONG_BUCKETS] = {0};

    afs::LongCon* d_cm = nullptr;       // EK / CARD with L <= 64, sorted by padded length
    uint32_t* d_cm_lits = nullptr;
    int32_t* d_cm_slots = nullptr;
    int32_t cm_begin[afs::CM_BUCKETS + 1] = {0};
    int32_t cm_maxL = 0;                // longest CMED constraint (rows of the shared-memory pmf buffer - 1)

    // original constraint index of every class entry, and (problems created with weights only) unit-weight twins of the
    // class records: the per-constraint gradient magnitudes (afs_constraint_grad_l1) are taken without the weights
    int32_t *d_pull_id = nullptr, *d_med_id = nullptr, *d_cm_id = nullptr, *d_long_id = nullptr;
    afs::MedCon* d_med_u = nullptr;
    afs::LongCon *d_cm_u = nullptr, *d_long_u = nullptr;
    bool unit_w_mode = false;           // the push launches of the current call read the unit-weight twins

    afs::CountCon* d_count = nullptr;   // all m constraints, original order
    uint32_t* d_count_lits = nullptr;

    int64_t n_pull = 0, n_med = 0, n_long = 0, n_cm = 0;
    afs::ResPlan res[afs::RES_PLANS];

    // the library's own second stream: per iteration the pull-clause counts (which need only the sign words of X_t)
    // run beside the variable pass; forked from and joined to the caller's stream with events, never synchronised
    cudaStream_t aux_stream = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;

    // ---- run state -----------------------------------------------------------------------------------------
    afs::Workspace ws;
    int64_t last_launches = 0;
    int32_t opt_mode = 0;
    int32_t retire_every = 32;          // streaming path: retire restarts at a fixed point every this many iterations (0 = never)
    int32_t last_resident = 0;
    afs::Profiler prof;
};
