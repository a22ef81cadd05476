// afs_problem.cu -- S0 of the path (host, once, untimed; "incurred once"): validation, bucketing by
// (type, length class), forward + transposed CSR, upload; and afs_coeffs (eq. 3 / Appendix A, PAPER.md L49-L52,
// L223-L255) with exact big-integer numerators.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <numeric>

#include "afs_internal.h"

using namespace afs;

#define CUDA_TRY(x)                          \
    do {                                     \
        cudaError_t e_ = (x);                \
        if (e_ != cudaSuccess) {             \
            afs::note_cuda_error(e_, __FILE__, __LINE__); \
            (void)cudaGetLastError();        \
            return AFS_ERR_CUDA;             \
        }                                    \
    } while (0)

template <typename T>
static afs_status upload(T** dst, const std::vector<T>& src)
{
    *dst = nullptr;
    size_t bytes = std::max<size_t>(src.size(), 1) * sizeof(T);
    if (cudaMalloc((void**)dst, bytes) != cudaSuccess) {
        (void)cudaGetLastError();
        return AFS_ERR_ALLOC;
    }
    if (!src.empty()) CUDA_TRY(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return AFS_OK;
}


// leave-one-out pmf indices that enter dFE/dy_j = sum_t d_t q_t^(-j), d_t = (sp_t - sp_{t+1})/2
static void long_targets(int type, int L, int k, LongCon& c)
{
    c.tA = c.tB = 0;
    c.wA = c.wB = 0.f;
    auto setA = [&](int t, float w) { if (t >= 0 && t <= L - 1) { c.tA = t; c.wA = w; } };
    auto setB = [&](int t, float w) { if (t >= 0 && t <= L - 1) { c.tB = t; c.wB = w; } };
    switch (type) {
    case AFS_OR: setA(0, 1.f); break;
    case AFS_EO: setA(0, 1.f); setB(1, -1.f); break;
    case AFS_AMO: setA(1, -1.f); break;
    case AFS_EK: setA(k - 1, 1.f); setB(k, -1.f); break;
    case AFS_CARD: setA(k - 1, 1.f); break;
    case AFS_NAE: setA(0, 1.f); setB(L - 1, -1.f); break;
    default: break;
    }
    if (c.wA != 0.f && c.wB != 0.f && c.tA == c.tB) {   // NAE with L = 1 cannot happen (rejected); keep safe anyway
        c.wA += c.wB; c.wB = 0.f;
    }
}

static afs_status create_impl(int32_t n_vars, int32_t n_cons, const int64_t* row_ptr, const int32_t* lits,
                              const int32_t* types, const int32_t* k, const float* weights, int32_t device,
                              afs_problem** out);

extern "C" afs_status afs_problem_create(int32_t n_vars, int32_t n_cons, const int64_t* row_ptr, const int32_t* lits,
                                         const int32_t* types, const int32_t* k, int32_t device, afs_problem** out)
{ return create_impl(n_vars, n_cons, row_ptr, lits, types, k, nullptr, device, out); }

extern "C" afs_status afs_problem_create_w(int32_t n_vars, int32_t n_cons, const int64_t* row_ptr, const int32_t* lits,
                                           const int32_t* types, const int32_t* k, const float* weights, int32_t device,
                                           afs_problem** out)
{
    if (weights)
        for (int c = 0; c < n_cons; ++c)
            if (!std::isfinite(weights[c])) { if (out) *out = nullptr; return AFS_ERR_INVALID_ARG; }
    return create_impl(n_vars, n_cons, row_ptr, lits, types, k, weights, device, out);
}

static afs_status create_impl(int32_t n_vars, int32_t n_cons, const int64_t* row_ptr, const int32_t* lits,
                              const int32_t* types, const int32_t* k, const float* weights, int32_t device,
                              afs_problem** out)
{
    if (!out) return AFS_ERR_INVALID_ARG;
    *out = nullptr;
    if (n_vars < 1 || n_cons < 0 || !row_ptr || (n_cons > 0 && (!lits || !types || !k))) return AFS_ERR_INVALID_ARG;
    if (row_ptr[0] != 0) return AFS_ERR_BAD_LITERAL;
    const int n = n_vars, m = n_cons;
    // ---------------------------------------------------------------- validation (G5, G6, G8)
    bool unsupported = false;
    {
        std::vector<int32_t> stamp(n, -1);
        for (int c = 0; c < m; ++c) {
            int64_t L = row_ptr[c + 1] - row_ptr[c];
            if (L < 1 || L > 0x3fffffff) return AFS_ERR_BAD_LITERAL;
            int ty = types[c];
            if (ty < 0 || ty > 6) return AFS_ERR_BAD_TYPE;
            if (ty == AFS_NAE && L < 2) return AFS_ERR_BAD_K;
            if ((ty == AFS_EK || ty == AFS_CARD) && (k[c] < 0 || k[c] > L + 1)) return AFS_ERR_BAD_K;
            if (ty == AFS_XOR && (k[c] < 0 || k[c] > 1)) return AFS_ERR_BAD_K;
            for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
                int32_t l = lits[e];
                if (l == 0 || l > n || l < -n) return AFS_ERR_BAD_LITERAL;
                int v = std::abs(l) - 1;
                if (stamp[v] == c) return AFS_ERR_DUP_VAR;
                stamp[v] = c;
            }
            if ((ty == AFS_EK || ty == AFS_CARD) && L > LONG_MAX_LEN) unsupported = true;
        }
    }
    if (unsupported) return AFS_ERR_UNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        (void)cudaGetLastError();
        return AFS_ERR_CUDA;
    }
    int prev_device = -1;
    if (cudaGetDevice(&prev_device) != cudaSuccess) { (void)cudaGetLastError(); prev_device = -1; }
    struct Restore { int d; ~Restore() { if (d >= 0) { cudaSetDevice(d); (void)cudaGetLastError(); } } } restore{prev_device};
    CUDA_TRY(cudaSetDevice(device));

    afs_problem* P = new (std::nothrow) afs_problem();
    if (!P) return AFS_ERR_ALLOC;
    P->n = n; P->m = m; P->nnz = row_ptr[m]; P->device = device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) P->sm_count = prop.multiProcessorCount;

    try {
        // ------------------------------------------------------------ classification
        enum { C_PULL = 0, C_MED = 1, C_LONG = 2, C_CMED = 3 };
        std::vector<uint8_t> cls(m);
        for (int c = 0; c < m; ++c) {
            int L = (int)(row_ptr[c + 1] - row_ptr[c]);
            int ty = types[c];
            bool prod = (ty == AFS_OR || ty == AFS_XOR);
            // a weighted short clause is materialised like any other constraint: the pull streams stay weight-free
            const bool unit_w = !weights || weights[c] == 1.0f;
            if ((prod || ty == AFS_NAE) && L <= PULL_MAX_LEN && unit_w) cls[c] = C_PULL;
            else if (prod || ty == AFS_NAE || ty == AFS_EO || ty == AFS_AMO) cls[c] = C_MED;   // any length
            else if ((ty == AFS_EK || ty == AFS_CARD) && L <= CM_MAX_LEN) cls[c] = C_CMED;
            else cls[c] = C_LONG;
        }
        // ------------------------------------------------------------ scratch slots, transposed-CSR order
        // slot order: by variable, then constraint id, then position (a stable counting sort over the forward CSR).
        // Two row ranges: the rows of MED / CMED literals first ([0, nslots_a), slot_ptr), then the rows of the LONG
        // class ([nslots_a, nslots), lslot_ptr): the latter are read through their own pass (k_glong), which takes
        // boundary literals' gradients from the per-(constraint, restart) pairs instead of the rows.
        auto is_long_cls = [&](int c) { return cls[c] == C_LONG; };
        std::vector<int32_t> slot_ptr(n + 1, 0), lslot_ptr(n + 1, 0);
        for (int c = 0; c < m; ++c)
            if (cls[c] != C_PULL)
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) (is_long_cls(c) ? lslot_ptr : slot_ptr)[std::abs(lits[e])]++;
        for (int v = 0; v < n; ++v) { slot_ptr[v + 1] += slot_ptr[v]; lslot_ptr[v + 1] += lslot_ptr[v]; }
        const int64_t nslots_a = slot_ptr[n];
        {   // slot ids, class offsets and run counts are 32-bit inside the kernels
            int64_t nonpull = 0;
            for (int c = 0; c < m; ++c) if (cls[c] != C_PULL) nonpull += row_ptr[c + 1] - row_ptr[c];
            if (nonpull > 0x7fffff00LL) { delete P; return AFS_ERR_UNSUPPORTED; }
        }
        P->nslots = nslots_a + lslot_ptr[n];
        P->nslots_a = nslots_a;
        std::vector<int32_t> fill(slot_ptr.begin(), slot_ptr.end() - 1), lfill(lslot_ptr.begin(), lslot_ptr.end() - 1);
        std::vector<int32_t> slot_of((size_t)P->nnz, -1);
        for (int c = 0; c < m; ++c)
            if (cls[c] != C_PULL)
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
                    const int v = std::abs(lits[e]) - 1;
                    slot_of[e] = is_long_cls(c) ? (int32_t)(nslots_a + lfill[v]++) : fill[v]++;
                }

        auto lit_word = [](int32_t l) -> uint32_t { return (uint32_t)(std::abs(l) - 1) | (l < 0 ? LIT_NEG : 0u); };

        // ------------------------------------------------------------ pull streams: runs of equal (kind, nother)
        if (n > MAX_VARS) { delete P; return AFS_ERR_UNSUPPORTED; }
        struct Occ { int c; int j; int key; };     // key = kind * 8 + nother
        std::vector<std::vector<Occ>> occs(n);
        std::vector<float> gconst(n, 0.f);
        std::vector<CountCon> pc;
        std::vector<uint32_t> pc_lits;
        std::vector<PullClause> pcp;
        std::vector<int32_t> pull_id, med_id, cm_id, long_id;   // original constraint index of every class entry
        for (int c = 0; c < m; ++c) {
            if (cls[c] != C_PULL) continue;
            P->n_pull++;
            pull_id.push_back(c);
            int L = (int)(row_ptr[c + 1] - row_ptr[c]);
            const int32_t* lc = lits + row_ptr[c];
            CountCon cc; cc.off = (int64_t)pc_lits.size(); cc.L = L; cc.type = (int16_t)types[c]; cc.pad = 0; cc.k = k[c]; cc.pad2 = 0;
            pc.push_back(cc);
            for (int j = 0; j < L; ++j) pc_lits.push_back(lit_word(lc[j]));
            int kind = types[c] == AFS_OR ? (int)PH_KIND_OR : types[c] == AFS_XOR ? (int)PH_KIND_XOR : (int)PH_KIND_NAE;
            PullClause pq{};
            pq.hdr = (uint32_t)L | ((uint32_t)kind << 3) | ((uint32_t)(k[c] & 1) << 5);
            for (int j = 0; j < L; ++j) pq.lit[j] = lit_word(lc[j]);
            pcp.push_back(pq);
            for (int j = 0; j < L; ++j) {
                int v = std::abs(lc[j]) - 1;
                bool sign = (lc[j] < 0) != (types[c] == AFS_XOR && !(k[c] & 1));
                if (L == 1) { gconst[v] += sign ? -1.f : 1.f; continue; }   // OR: dFE/dy = 1; XOR: +-1
                occs[v].push_back({c, j, kind * 8 + (L - 1)});
            }
        }
        std::vector<int32_t> pull_ptr(n + 1, 0), run_ptr(n + 1, 0);
        std::vector<uint32_t> pull_words, runs;
        for (int v = 0; v < n; ++v) {
            auto& ov = occs[v];
            std::stable_sort(ov.begin(), ov.end(), [](const Occ& a, const Occ& b) { return a.key < b.key; });
            size_t i = 0;
            while (i < ov.size()) {
                size_t e = i;
                while (e < ov.size() && ov[e].key == ov[i].key) ++e;
                int kind = ov[i].key / 8, nother = ov[i].key % 8;
                if (e - i > 0x07ffffffu) { delete P; return AFS_ERR_UNSUPPORTED; }   // 27-bit run count
                runs.push_back(((uint32_t)kind << 30) | ((uint32_t)nother << 27) | (uint32_t)(e - i));
                for (; i < e; ++i) {
                    int c = ov[i].c, j = ov[i].j;
                    int L = (int)(row_ptr[c + 1] - row_ptr[c]);
                    const int32_t* lc = lits + row_ptr[c];
                    bool sign = (lc[j] < 0) != (types[c] == AFS_XOR && !(k[c] & 1));
                    bool first = true;
                    for (int q = 0; q < L; ++q) {
                        if (q == j) continue;
                        pull_words.push_back((uint32_t)(std::abs(lc[q]) - 1) | (lc[q] < 0 ? PE_NEG : 0u) |
                                             ((first && sign) ? PE_SIGN : 0u));
                        first = false;
                    }
                }
            }
            if (pull_words.size() > 0x7fffff00u) { delete P; return AFS_ERR_UNSUPPORTED; }
            pull_ptr[v + 1] = (int32_t)pull_words.size();
            run_ptr[v + 1] = (int32_t)runs.size();
        }
        occs.clear(); occs.shrink_to_fit();
        pull_words.resize(pull_words.size() + 32, 0u);   // staged chunk loads may read up to 31 entries past a stream
        P->pull_words = pull_ptr[n];
        // ------------------------------------------------------------ medium constraints (sorted by padded length)
        std::vector<MedCon> med;
        std::vector<uint32_t> med_lits;
        std::vector<int32_t> med_slots;
        {
            std::vector<int> ids;
            for (int c = 0; c < m; ++c) if (cls[c] == C_MED) ids.push_back(c);
            // longest first: the grid-stride loops and the resident kernel's work counter take the heavy ones early
            std::stable_sort(ids.begin(), ids.end(), [&](int a, int b) {
                return (row_ptr[a + 1] - row_ptr[a]) > (row_ptr[b + 1] - row_ptr[b]);
            });
            for (size_t i = 0; i < ids.size(); ++i) {
                int c = ids[i];
                MedCon mc;
                int64_t L = row_ptr[c + 1] - row_ptr[c];
                mc.off = (int32_t)med_lits.size(); mc.L = (int32_t)L;
                mc.type = types[c]; mc.k = k[c]; mc.w = weights ? weights[c] : 1.0f;
                if (types[c] != AFS_OR && types[c] != AFS_XOR) P->med_two = true;
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
                    med_lits.push_back(lit_word(lits[e]));
                    med_slots.push_back(slot_of[e]);
                }
                med.push_back(mc);
                med_id.push_back(c);
            }
            P->med_nnz = (int64_t)med_lits.size();
            P->n_med = (int64_t)ids.size();
        }
        // ------------------------------------------------------------ long constraints (sorted by row count, longest first)
        std::vector<LongCon> lng, cmv;
        std::vector<uint32_t> long_lits, cm_lits;
        std::vector<int32_t> long_slots, cm_slots;
        auto build_count_class = [&](int want_cls, auto bucket_fn, int nbuckets, int32_t* begin, int32_t* maxL,
                                     std::vector<LongCon>& out, std::vector<uint32_t>& olits, std::vector<int32_t>& oslots,
                                     std::vector<int32_t>& oid) {
            std::vector<int> ids;
            for (int c = 0; c < m; ++c) if (cls[c] == want_cls) ids.push_back(c);
            std::stable_sort(ids.begin(), ids.end(), [&](int a, int b) {
                int ra = bucket_fn(a), rb = bucket_fn(b);
                if (ra != rb) return ra < rb;
                return (row_ptr[a + 1] - row_ptr[a]) > (row_ptr[b + 1] - row_ptr[b]);
            });
            int cur = 0;
            begin[0] = 0;
            for (size_t i = 0; i < ids.size(); ++i) {
                int c = ids[i];
                int bk = bucket_fn(c);
                while (cur < bk) begin[++cur] = (int32_t)i;
                LongCon lc;
                lc.off = (int32_t)olits.size(); lc.L = (int32_t)(row_ptr[c + 1] - row_ptr[c]);
                lc.type = types[c]; lc.k = k[c]; lc.w = weights ? weights[c] : 1.0f;
                long_targets(lc.type, lc.L, lc.k, lc);
                if (maxL) maxL[bk] = std::max(maxL[bk], lc.L);
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
                    olits.push_back(lit_word(lits[e]));
                    oslots.push_back(slot_of[e]);
                }
                out.push_back(lc);
                oid.push_back(c);
            }
            while (cur < nbuckets) begin[++cur] = (int32_t)ids.size();
            return (int64_t)ids.size();
        };
        P->n_long = build_count_class(C_LONG, [&](int c) { return (int)((row_ptr[c + 1] - row_ptr[c] + 1 + 127) / 128) - 1; },
                                      LONG_BUCKETS, P->long_begin, P->long_maxL, lng, long_lits, long_slots, long_id);
        P->n_cm = build_count_class(C_CMED, [&](int c) { return (int)((row_ptr[c + 1] - row_ptr[c] + 15) / 16) - 1; },
                                    CM_BUCKETS, P->cm_begin, nullptr, cmv, cm_lits, cm_slots, cm_id);
        for (const LongCon& x : cmv) P->cm_maxL = std::max(P->cm_maxL, x.L);
        // ------------------------------------------------------------ generic forward CSR for the count-only kernel
        std::vector<CountCon> cnt(m);
        std::vector<uint32_t> cnt_lits((size_t)P->nnz);
        for (int c = 0; c < m; ++c) {
            cnt[c].off = row_ptr[c]; cnt[c].L = (int32_t)(row_ptr[c + 1] - row_ptr[c]);
            cnt[c].type = (int16_t)types[c]; cnt[c].pad = 0; cnt[c].k = k[c]; cnt[c].pad2 = 0;
        }
        for (int64_t e = 0; e < P->nnz; ++e) cnt_lits[e] = lit_word(lits[e]);

        afs_status st = AFS_OK;
        auto up = [&](auto** dst, const auto& src) { if (st == AFS_OK) st = upload(dst, src); };
        // ------------------------------------------------------------ plans of the tile-resident kernel
        if (lng.empty()) {
            std::vector<double> vcost(n);
            for (int v = 0; v < n; ++v)
                // warp-instructions, from the source-level counts of the resident kernel: ~10 per staged pull word,
                // ~30 per run, ~60 per variable, plus the P3 share (~8 per gradient row)
                vcost[v] = 10.0 * (pull_ptr[v + 1] - pull_ptr[v]) + 30.0 * (run_ptr[v + 1] - run_ptr[v]) +
                           8.0 * (slot_ptr[v + 1] - slot_ptr[v]) + 60.0;
            struct It { double cost; ResItem it; bool cm; };
            std::vector<It> its;
            for (size_t i = 0; i < med.size(); ++i) {
                its.push_back({40.0 + 30.0 * med[i].L, ResItem{0u, (uint32_t)i}, false});
            }
            for (size_t i = 0; i < cmv.size(); ++i) {
                const double L = cmv[i].L;
                const double chain = std::max({(double)cmv[i].tA, (double)cmv[i].tB, L - 1 - cmv[i].tA, L - 1 - cmv[i].tB}) + 1;
                // forward pmf ~4.2 per cell (L^2 / 2 cells), chains ~5 per step and pair of literals, ~50 per literal
                its.push_back({2.1 * L * L + L * (50.0 + 2.5 * chain), ResItem{0u, (uint32_t)i}, true});
            }
            std::stable_sort(its.begin(), its.end(), [](const It& x, const It& y) { return x.cost > y.cost; });
            for (int pi = 0; pi < RES_PLANS; ++pi) {
                const int C = pi + 1;
                ResPlan& rp = P->res[pi];
                rp.C = C;
                std::vector<int32_t> vbeg(C + 1, 0), ibeg(C + 1, 0), pbeg(C + 1, 0);
                double tot = std::accumulate(vcost.begin(), vcost.end(), 0.0), acc = 0.0;
                int r = 1;
                for (int v = 0; v < n && r < C; ++v) {
                    acc += vcost[v];
                    while (r < C && acc >= tot * r / C) vbeg[r++] = v + 1;
                }
                while (r < C) vbeg[r++] = n;
                vbeg[C] = n;
                std::vector<std::vector<ResItem>> per(C);
                std::vector<std::vector<int32_t>> perc(C);
                std::vector<double> load(C, 0.0);
                for (const It& x : its) {   // longest processing time first, onto the least loaded rank
                    int best = (int)(std::min_element(load.begin(), load.end()) - load.begin());
                    if (x.cm) perc[best].push_back((int32_t)x.it.idx); else per[best].push_back(x.it);
                    load[best] += x.cost;
                }
                std::vector<ResItem> flat;
                std::vector<int32_t> cflat, cbeg(C + 1, 0);
                for (int q = 0; q < C; ++q) {
                    ibeg[q] = (int32_t)flat.size();
                    flat.insert(flat.end(), per[q].begin(), per[q].end());
                    cbeg[q] = (int32_t)cflat.size();
                    cflat.insert(cflat.end(), perc[q].begin(), perc[q].end());
                }
                ibeg[C] = (int32_t)flat.size();
                cbeg[C] = (int32_t)cflat.size();
                for (int q = 0; q < C; ++q) {
                    int plits = 0;
                    for (const ResItem& it : per[q]) plits += med[it.idx].L;
                    for (int32_t ci : perc[q]) plits += cmv[ci].L;
                    rp.cap_words = std::max(rp.cap_words, pull_ptr[vbeg[q + 1]] - pull_ptr[vbeg[q]] + 32);
                    rp.cap_runs = std::max(rp.cap_runs, run_ptr[vbeg[q + 1]] - run_ptr[vbeg[q]]);
                    rp.cap_own = std::max(rp.cap_own, vbeg[q + 1] - vbeg[q]);
                    rp.cap_plits = std::max(rp.cap_plits, plits);
                    rp.cap_cm = std::max(rp.cap_cm, (int)perc[q].size());
                    rp.cap_push = std::max(rp.cap_push, (int)per[q].size());
                }
                up(&rp.d_cm_begin, cbeg);
                up(&rp.d_cm_items, cflat);
                for (int q = 0; q <= C; ++q) pbeg[q] = (int32_t)((int64_t)pc.size() * q / C);
                up(&rp.d_var_begin, vbeg);
                up(&rp.d_item_begin, ibeg);
                up(&rp.d_items, flat);
                up(&rp.d_pc_begin, pbeg);
            }
        }
        up(&P->d_pull_ptr, pull_ptr);
        up(&P->d_pull_words, pull_words);
        up(&P->d_run_ptr, run_ptr);
        up(&P->d_runs, runs);
        up(&P->d_pull_gconst, gconst);
        up(&P->d_pc, pc);
        up(&P->d_pc_lits, pc_lits);
        up(&P->d_pcp, pcp);
        up(&P->d_slot_ptr, slot_ptr);
        {   // per LONG-class row (in lslot order): (index in d_long) << 1 | literal negated
            std::vector<int32_t> lslot_info((size_t)lslot_ptr[n], 0);
            for (size_t i = 0; i < lng.size(); ++i)
                for (int j = 0; j < lng[i].L; ++j)
                    lslot_info[long_slots[lng[i].off + j] - nslots_a] = (int32_t)((i << 1) | (long_lits[lng[i].off + j] >> 31));
            up(&P->d_lslot_info, lslot_info);
            up(&P->d_lslot_ptr, lslot_ptr);
        }
        up(&P->d_med, med);
        up(&P->d_med_lits, med_lits);
        up(&P->d_med_slots, med_slots);
        up(&P->d_long, lng);
        up(&P->d_long_lits, long_lits);
        up(&P->d_long_slots, long_slots);
        P->long_nnz = (int64_t)long_lits.size();
        {
            std::vector<int32_t> goff(lng.size() + 1, 0);
            for (size_t i = 0; i < lng.size(); ++i) goff[i + 1] = goff[i] + (lng[i].L + 31) / 32;
            P->long_grows = goff[lng.size()];
            up(&P->d_long_goff, goff);
        }
        up(&P->d_long_f, lng);
        up(&P->d_long_lits_f, long_lits);
        up(&P->d_long_slots_f, long_slots);
        up(&P->d_cm, cmv);
        up(&P->d_cm_lits, cm_lits);
        up(&P->d_cm_slots, cm_slots);
        up(&P->d_pull_id, pull_id); up(&P->d_med_id, med_id); up(&P->d_cm_id, cm_id); up(&P->d_long_id, long_id);
        if (weights) {   // unit-weight twins of the class records, for the per-constraint gradient magnitudes
            std::vector<MedCon> med_u(med); for (auto& x : med_u) x.w = 1.0f;
            std::vector<LongCon> cm_u(cmv), lng_u(lng);
            for (auto& x : cm_u) x.w = 1.0f;
            for (auto& x : lng_u) x.w = 1.0f;
            up(&P->d_med_u, med_u); up(&P->d_cm_u, cm_u); up(&P->d_long_u, lng_u);
        }
        up(&P->d_count, cnt);
        up(&P->d_count_lits, cnt_lits);
        if (st != AFS_OK) { afs_problem_destroy(P); return st; }
        if (cudaStreamCreateWithFlags(&P->aux_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&P->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&P->ev_join, cudaEventDisableTiming) != cudaSuccess) {
            (void)cudaGetLastError();
            afs_problem_destroy(P);
            return AFS_ERR_CUDA;
        }
        CUDA_TRY(cudaDeviceSynchronize());
    } catch (const std::bad_alloc&) {
        afs_problem_destroy(P);
        return AFS_ERR_ALLOC;
    }
    *out = P;
    return AFS_OK;
}

namespace afs { void free_workspace(afs_problem* p); }

extern "C" void afs_problem_destroy(afs_problem* p)
{
    if (!p) return;
    int prev_device = -1;
    if (cudaGetDevice(&prev_device) != cudaSuccess) { (void)cudaGetLastError(); prev_device = -1; }
    cudaSetDevice(p->device);
    cudaDeviceSynchronize();
    cudaFree(p->d_pull_ptr); cudaFree(p->d_pull_words); cudaFree(p->d_slot_ptr); cudaFree(p->d_lslot_info); cudaFree(p->d_lslot_ptr);
    cudaFree(p->d_pull_id); cudaFree(p->d_med_id); cudaFree(p->d_cm_id); cudaFree(p->d_long_id);
    cudaFree(p->d_med_u); cudaFree(p->d_cm_u); cudaFree(p->d_long_u);
    cudaFree(p->d_run_ptr); cudaFree(p->d_runs); cudaFree(p->d_pull_gconst); cudaFree(p->d_pc); cudaFree(p->d_pc_lits); cudaFree(p->d_pcp);
    cudaFree(p->d_med); cudaFree(p->d_med_lits); cudaFree(p->d_med_slots);
    cudaFree(p->d_long); cudaFree(p->d_long_lits); cudaFree(p->d_long_slots);
    cudaFree(p->d_long_goff); cudaFree(p->d_long_f); cudaFree(p->d_long_lits_f); cudaFree(p->d_long_slots_f);
    cudaFree(p->d_cm); cudaFree(p->d_cm_lits); cudaFree(p->d_cm_slots);
    cudaFree(p->d_count); cudaFree(p->d_count_lits);
    for (int i = 0; i < afs::RES_PLANS; ++i) {
        cudaFree(p->res[i].d_var_begin); cudaFree(p->res[i].d_item_begin);
        cudaFree(p->res[i].d_items); cudaFree(p->res[i].d_pc_begin);
        cudaFree(p->res[i].d_cm_begin); cudaFree(p->res[i].d_cm_items);
    }
    afs::free_workspace(p);
    if (p->aux_stream) cudaStreamDestroy(p->aux_stream);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    for (cudaEvent_t e : p->prof.pool) cudaEventDestroy(e);
    cudaFree(p->prof.d_work);
    (void)cudaGetLastError();
    delete p;
    if (prev_device >= 0) { cudaSetDevice(prev_device); (void)cudaGetLastError(); }
}

extern "C" int64_t afs_problem_info(const afs_problem* p, int32_t what)
{
    if (!p) return -1;
    switch (what) {
    case 0: return p->n;
    case 1: return p->m;
    case 2: return p->nnz;
    case 3: return p->n_pull;
    case 4: return p->n_med;
    case 5: return p->n_long + p->n_cm;
    case 6: return p->nslots;
    case 7: return p->last_launches;
    case 8: return (int64_t)p->ws.bytes;
    case 9: return p->last_resident;
    default: return -1;
    }
}

extern "C" afs_status afs_set_option(afs_problem* p, int32_t what, int64_t value)
{
    if (!p) return AFS_ERR_INVALID_ARG;
    if (what == 0 && value >= 0 && value <= 2) { p->opt_mode = (int32_t)value; return AFS_OK; }
    if (what == 1 && value >= 0 && value <= (1 << 20)) { p->prof.stride = (int)value; return AFS_OK; }
    if (what == 2 && value >= 0 && value <= (1 << 20)) { p->retire_every = (int32_t)value; return AFS_OK; }
    return AFS_ERR_INVALID_ARG;
}

extern "C" const char* afs_status_string(afs_status s)
{
    switch (s) {
    case AFS_OK: return "ok";
    case AFS_ERR_INVALID_ARG: return "invalid argument";
    case AFS_ERR_BAD_TYPE: return "constraint type out of range";
    case AFS_ERR_BAD_K: return "threshold k out of range for this constraint";
    case AFS_ERR_BAD_LITERAL: return "bad literal, empty constraint or malformed row_ptr";
    case AFS_ERR_DUP_VAR: return "variable repeated inside a constraint";
    case AFS_ERR_ALLOC: return "allocation failed";
    case AFS_ERR_CUDA: return "CUDA error or no CUDA device";
    case AFS_ERR_UNSUPPORTED: return "unsupported by this build";
    case AFS_ERR_STATIC_LIMIT: return "n and B exceed the static scratch array (AFS_STATIC_SCRATCH_BYTES) of afs_round_count_static";
    default: return "unknown status";
    }
}

extern "C" int32_t afs_abi_version(void) { return AFS_ABI_VERSION; }

namespace afs {
static thread_local char g_last_error[256] = "";
void note_cuda_error(cudaError_t e, const char* file, int line)
{
    const char* base = file;
    for (const char* c = file; *c; ++c) if (*c == '/') base = c + 1;
    snprintf(g_last_error, sizeof(g_last_error), "%s (%s:%d)", cudaGetErrorString(e), base, line);
}
}  // namespace afs

extern "C" const char* afs_last_error_message(void) { return afs::g_last_error; }

// =====================================================================================================================
// afs_coeffs: eq. (3) through the Appendix-A closed forms (L223-L255; G2-G5).
// The integer coefficients of (1+rho)^a (1-rho)^b are Krawtchouk values with heavy cancellation, so they are built
// exactly, in fixed-width two's-complement big integers, by repeated multiplication with (1 +- rho).
// =====================================================================================================================
namespace {

struct Big {   // two's complement, little-endian 64-bit limbs, fixed width
    std::vector<uint64_t> w;
    explicit Big(int limbs = 1, int64_t v = 0) : w(limbs, v < 0 ? ~0ull : 0ull) { w[0] = (uint64_t)v; }
    bool neg() const { return (w.back() >> 63) != 0; }
    void add(const Big& o) {
        unsigned __int128 c = 0;
        for (size_t i = 0; i < w.size(); ++i) { c += (unsigned __int128)w[i] + o.w[i]; w[i] = (uint64_t)c; c >>= 64; }
    }
    void sub(const Big& o) {
        unsigned __int128 c = 1;
        for (size_t i = 0; i < w.size(); ++i) { c += (unsigned __int128)w[i] + (uint64_t)~o.w[i]; w[i] = (uint64_t)c; c >>= 64; }
    }
    void negate() { Big z((int)w.size(), 0); z.sub(*this); w.swap(z.w); }
    void mul_small(int64_t f) {   // |f| < 2^31
        bool fl = f < 0; uint64_t a = (uint64_t)(fl ? -f : f);
        bool sg = neg(); if (sg) negate();
        unsigned __int128 c = 0;
        for (size_t i = 0; i < w.size(); ++i) { c += (unsigned __int128)w[i] * a; w[i] = (uint64_t)c; c >>= 64; }
        if (sg != fl) negate();
    }
    // value = mant * 2^exp, mant carries the top 64 bits (relative error < 2^-63)
    void to_ld(long double& mant, int& exp) const {
        Big t = *this; bool sg = t.neg(); if (sg) t.negate();
        int top = (int)t.w.size() - 1;
        while (top > 0 && t.w[top] == 0) --top;
        if (t.w[top] == 0) { mant = 0.0L; exp = 0; return; }
        int lz = __builtin_clzll(t.w[top]);
        uint64_t hi = t.w[top] << lz;
        if (lz && top > 0) hi |= t.w[top - 1] >> (64 - lz);
        mant = (long double)hi; exp = top * 64 - lz;
        if (sg) mant = -mant;
    }
};

// num / (den * 2^shift) as a double
double ratio(const Big& num, const Big& den, int shift)
{
    long double mn, md; int en, ed;
    num.to_ld(mn, en); den.to_ld(md, ed);
    if (mn == 0.0L) return 0.0;
    return (double)ldexpl(mn / md, en - ed - shift);
}

}  // namespace

extern "C" afs_status afs_coeffs(int32_t type, int32_t L, int32_t k, double* a)
{
    if (!a || L < 1 || L > 4096) return AFS_ERR_INVALID_ARG;
    if (type < 0 || type > 6) return AFS_ERR_BAD_TYPE;
    if (type == AFS_NAE && L < 2) return AFS_ERR_BAD_K;
    if ((type == AFS_EK || type == AFS_CARD) && (k < 0 || k > L + 1)) return AFS_ERR_BAD_K;
    if (type == AFS_XOR && (k < 0 || k > 1)) return AFS_ERR_BAD_K;
    const int n = L;
    auto pow2m = [](int e) { return std::ldexp(1.0, -e); };   // 2^-e (0 on underflow)
    for (int s = 0; s <= n; ++s) a[s] = 0.0;
    try {
        switch (type) {
        case AFS_OR:    // L225: a_0 = 2^-(n-1) - 1, a_s = 2^-(n-1)
            for (int s = 1; s <= n; ++s) a[s] = pow2m(n - 1);
            a[0] = pow2m(n - 1) - 1.0;
            return AFS_OK;
        case AFS_EO:    // L229: a_0 = 1 - n 2^-(n-1), a_s = (2s - n) 2^-(n-1)
            for (int s = 1; s <= n; ++s) a[s] = std::ldexp((double)(2 * s - n), -(n - 1));
            a[0] = 1.0 - std::ldexp((double)n, -(n - 1));
            return AFS_OK;
        case AFS_AMO:   // L237 with the constant term repaired (G3): a_0 = 1 - (n+1) 2^-(n-1), a_s = (2s - n - 1) 2^-(n-1)
            for (int s = 1; s <= n; ++s) a[s] = std::ldexp((double)(2 * s - n - 1), -(n - 1));
            a[0] = 1.0 - std::ldexp((double)(n + 1), -(n - 1));
            return AFS_OK;
        case AFS_NAE:   // L243: a_0 = 2^-(n-2) - 1, a_s = 2^-(n-2) for even s, 0 for odd s
            for (int s = 2; s <= n; s += 2) a[s] = pow2m(n - 2);
            a[0] = pow2m(n - 2) - 1.0;
            return AFS_OK;
        case AFS_XOR:   // L249 (G2): a_n = +1 for odd parity, -1 for even parity
            a[n] = (k & 1) ? 1.0 : -1.0;
            return AFS_OK;
        default: break;
        }
        // ---- EK / CARD: degenerate thresholds first (G4, G5)
        if (type == AFS_CARD && k == 0) { a[0] = -1.0; return AFS_OK; }
        if (k == n + 1) { a[0] = 1.0; return AFS_OK; }
        if (type == AFS_EK && k == 0) {           // "no literal true" = NOT OR:  a = -a_OR
            for (int s = 1; s <= n; ++s) a[s] = -pow2m(n - 1);
            a[0] = 1.0 - pow2m(n - 1);
            return AFS_OK;
        }
        if (type == AFS_EK && k == n) {           // "all true": f(y) = -OR(-y), a_s = -(-1)^s a_s^OR
            for (int s = 1; s <= n; ++s) a[s] = ((s & 1) ? 1.0 : -1.0) * pow2m(n - 1);
            a[0] = 1.0 - pow2m(n - 1);
            return AFS_OK;
        }
        const int limbs = (n + 64) / 64 + 2;
        // Pascal rows C(n, .) and C(n-1, .)
        auto pascal = [&](int N) {
            std::vector<Big> row(N + 1, Big(limbs, 0));
            row[0] = Big(limbs, 1);
            for (int r = 1; r <= N; ++r)
                for (int i = r; i >= 1; --i) row[i].add(row[i - 1]);
            return row;
        };
        std::vector<Big> Cn = pascal(n), Cn1 = pascal(n - 1);
        // poly = (1+rho)^A (1-rho)^Bm
        const int A = type == AFS_CARD ? n - k : n - k - 1;
        const int Bm = k - 1;
        std::vector<Big> poly(A + Bm + 2, Big(limbs, 0));
        poly[0] = Big(limbs, 1);
        int deg = 0;
        for (int r = 0; r < A; ++r) { for (int i = deg + 1; i >= 1; --i) poly[i].add(poly[i - 1]); ++deg; }
        for (int r = 0; r < Bm; ++r) { for (int i = deg + 1; i >= 1; --i) poly[i].sub(poly[i - 1]); ++deg; }
        Big one(limbs, 1);
        if (type == AFS_CARD) {
            // L253-L255: a_0 = 1 - sum_{i>=k} C(n,i) / 2^(n-1);  a_s = C(n-1,k-1) [rho^(s-1)] poly / (C(n-1,s-1) 2^(n-1))
            Big S(limbs, 0);
            for (int i = k; i <= n; ++i) S.add(Cn[i]);
            Big P2(limbs, 0); P2.w[(n - 1) / 64] = 1ull << ((n - 1) % 64);
            P2.sub(S);
            a[0] = ratio(P2, one, n - 1);
            long double mc; int ec; Cn1[k - 1].to_ld(mc, ec);
            for (int s = 1; s <= n; ++s) {
                long double mn, md; int en, ed;
                poly[s - 1].to_ld(mn, en); Cn1[s - 1].to_ld(md, ed);
                a[s] = mn == 0.0L ? 0.0 : (double)ldexpl(mc * mn / md, ec + en - ed - (n - 1));
            }
        } else {
            // L233 as repaired (G4), 1 <= k <= n-1:  a_0 = 1 - C(n,k)/2^(n-1);
            // a_s = (C(n,k)/n) [rho^(s-1)] ((2k-n) + n rho) poly / (C(n-1,s-1) 2^(n-1)),  poly = (1+rho)^(n-k-1)(1-rho)^(k-1)
            long double mc; int ec; Cn[k].to_ld(mc, ec);
            a[0] = (double)(1.0L - ldexpl(mc, ec - (n - 1)));
            for (int s = 1; s <= n; ++s) {
                Big t(limbs, 0);
                if (s - 1 <= deg) { t = poly[s - 1]; t.mul_small(2 * k - n); }
                if (s - 2 >= 0 && s - 2 <= deg) { Big u = poly[s - 2]; u.mul_small(n); t.add(u); }
                long double mn, md; int en, ed;
                t.to_ld(mn, en); Cn1[s - 1].to_ld(md, ed);
                a[s] = mn == 0.0L ? 0.0 : (double)ldexpl(mc * mn / md / (long double)n, ec + en - ed - (n - 1));
            }
        }
    } catch (const std::bad_alloc&) {
        return AFS_ERR_ALLOC;
    }
    return AFS_OK;
}
