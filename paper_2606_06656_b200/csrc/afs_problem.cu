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

static int med_bucket(int64_t L) { return L <= 8 ? 0 : L <= 16 ? 1 : L <= 32 ? 2 : L <= 64 ? 3 : 4; }

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

extern "C" afs_status afs_problem_create(int32_t n_vars, int32_t n_cons, const int64_t* row_ptr, const int32_t* lits,
                                         const int32_t* types, const int32_t* k, int32_t device, afs_problem** out)
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
            bool count_type = !(ty == AFS_OR || ty == AFS_XOR);
            if (count_type && L > LONG_MAX_LEN) unsupported = true;
        }
    }
    if (unsupported) return AFS_ERR_UNSUPPORTED;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        (void)cudaGetLastError();
        return AFS_ERR_CUDA;
    }
    CUDA_TRY(cudaSetDevice(device));

    afs_problem* P = new (std::nothrow) afs_problem();
    if (!P) return AFS_ERR_ALLOC;
    P->n = n; P->m = m; P->nnz = row_ptr[m]; P->device = device;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) == cudaSuccess) P->sm_count = prop.multiProcessorCount;

    try {
        // ------------------------------------------------------------ classification
        enum { C_PULL = 0, C_MED = 1, C_LONG = 2 };
        std::vector<uint8_t> cls(m);
        for (int c = 0; c < m; ++c) {
            int L = (int)(row_ptr[c + 1] - row_ptr[c]);
            int ty = types[c];
            bool prod = (ty == AFS_OR || ty == AFS_XOR);
            if ((prod || ty == AFS_NAE) && L <= PULL_MAX_LEN) cls[c] = C_PULL;
            else if (prod) cls[c] = C_MED;   // any length: beyond MED_MAX_PROD the two-pass product kernel takes it
            else if ((ty == AFS_NAE || ty == AFS_EO || ty == AFS_AMO) && L <= MED_MAX_TWO) cls[c] = C_MED;
            else cls[c] = C_LONG;
        }
        // ------------------------------------------------------------ scratch slots, transposed-CSR order
        // slot order: by variable, then constraint id, then position (a stable counting sort over the forward CSR)
        std::vector<int32_t> slot_ptr(n + 1, 0);
        for (int c = 0; c < m; ++c)
            if (cls[c] != C_PULL)
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) slot_ptr[std::abs(lits[e])]++;
        for (int v = 0; v < n; ++v) slot_ptr[v + 1] += slot_ptr[v];
        P->nslots = slot_ptr[n];
        std::vector<int32_t> fill(slot_ptr.begin(), slot_ptr.end() - 1);
        std::vector<int32_t> slot_of((size_t)P->nnz, -1);
        for (int c = 0; c < m; ++c)
            if (cls[c] != C_PULL)
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) slot_of[e] = fill[std::abs(lits[e]) - 1]++;

        auto lit_word = [](int32_t l) -> uint32_t { return (uint32_t)(std::abs(l) - 1) | (l < 0 ? LIT_NEG : 0u); };

        // ------------------------------------------------------------ pull streams
        std::vector<int32_t> pull_ptr(n + 1, 0);
        for (int c = 0; c < m; ++c)
            if (cls[c] == C_PULL) {
                int L = (int)(row_ptr[c + 1] - row_ptr[c]);
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) pull_ptr[std::abs(lits[e])] += L;  // header + L-1
                P->n_pull++;
            }
        for (int v = 0; v < n; ++v) {
            int64_t s = (int64_t)pull_ptr[v + 1] + pull_ptr[v];
            if (s > 0x7fffffff) { delete P; return AFS_ERR_UNSUPPORTED; }
            pull_ptr[v + 1] = (int32_t)s;
        }
        P->pull_words = pull_ptr[n];
        std::vector<uint32_t> pull_words((size_t)P->pull_words);
        {
            std::vector<int32_t> pf(pull_ptr.begin(), pull_ptr.end() - 1);
            for (int c = 0; c < m; ++c) {
                if (cls[c] != C_PULL) continue;
                int L = (int)(row_ptr[c + 1] - row_ptr[c]);
                const int32_t* lc = lits + row_ptr[c];
                uint32_t kind = types[c] == AFS_OR ? PH_KIND_OR : types[c] == AFS_XOR ? PH_KIND_XOR : PH_KIND_NAE;
                for (int j = 0; j < L; ++j) {
                    int v = std::abs(lc[j]) - 1;
                    int32_t& w = pf[v];
                    uint32_t hdr = kind | ((uint32_t)(L - 1) << 2) | (lc[j] < 0 ? 32u : 0u) | (j == 0 ? 64u : 0u) |
                                   ((types[c] == AFS_XOR && (k[c] & 1)) ? 128u : 0u);
                    pull_words[w++] = hdr;
                    for (int i = 0; i < L; ++i)
                        if (i != j) pull_words[w++] = lit_word(lc[i]);
                }
            }
        }
        // ------------------------------------------------------------ medium constraints (sorted by padded length)
        std::vector<MedCon> med;
        std::vector<uint32_t> med_lits;
        std::vector<int32_t> med_slots;
        {
            std::vector<int> ids;
            for (int c = 0; c < m; ++c) if (cls[c] == C_MED) ids.push_back(c);
            auto bucket_of = [&](int c) { return med_bucket(row_ptr[c + 1] - row_ptr[c]); };
            std::stable_sort(ids.begin(), ids.end(), [&](int a, int b) {
                int ba = bucket_of(a), bb = bucket_of(b);
                if (ba != bb) return ba < bb;
                return types[a] < types[b];     // homogeneous warps inside a bucket
            });
            int cur = 0;
            P->med_begin[0] = 0;
            for (size_t i = 0; i < ids.size(); ++i) {
                int c = ids[i];
                int bk = bucket_of(c);
                while (cur < bk) P->med_begin[++cur] = (int32_t)i;
                MedCon mc;
                int64_t L = row_ptr[c + 1] - row_ptr[c];
                mc.off = (int32_t)med_lits.size(); mc.L = (int32_t)L;
                mc.type = types[c]; mc.k = k[c];
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
                    med_lits.push_back(lit_word(lits[e]));
                    med_slots.push_back(slot_of[e]);
                }
                med.push_back(mc);
            }
            while (cur < MED_BUCKETS) P->med_begin[++cur] = (int32_t)ids.size();
            P->n_med = (int64_t)ids.size();
        }
        // ------------------------------------------------------------ long constraints (sorted by row count, longest first)
        std::vector<LongCon> lng;
        std::vector<uint32_t> long_lits;
        std::vector<int32_t> long_slots;
        {
            std::vector<int> ids;
            for (int c = 0; c < m; ++c) if (cls[c] == C_LONG) ids.push_back(c);
            auto nr_of = [&](int c) { return (int)((row_ptr[c + 1] - row_ptr[c] + 1 + 127) / 128); };   // rows for q_0..q_L
            std::stable_sort(ids.begin(), ids.end(), [&](int a, int b) {
                int ra = nr_of(a), rb = nr_of(b);
                if (ra != rb) return ra < rb;
                return (row_ptr[a + 1] - row_ptr[a]) > (row_ptr[b + 1] - row_ptr[b]);
            });
            int cur = 0;
            P->long_begin[0] = 0;
            for (size_t i = 0; i < ids.size(); ++i) {
                int c = ids[i];
                int bk = nr_of(c) - 1;
                while (cur < bk) P->long_begin[++cur] = (int32_t)i;
                LongCon lc;
                lc.off = (int32_t)long_lits.size(); lc.L = (int32_t)(row_ptr[c + 1] - row_ptr[c]);
                lc.type = types[c]; lc.k = k[c];
                long_targets(lc.type, lc.L, lc.k, lc);
                P->long_maxL[bk] = std::max(P->long_maxL[bk], lc.L);
                for (int64_t e = row_ptr[c]; e < row_ptr[c + 1]; ++e) {
                    long_lits.push_back(lit_word(lits[e]));
                    long_slots.push_back(slot_of[e]);
                }
                lng.push_back(lc);
            }
            while (cur < LONG_BUCKETS) P->long_begin[++cur] = (int32_t)ids.size();
            P->n_long = (int64_t)ids.size();
        }
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
        up(&P->d_pull_ptr, pull_ptr);
        up(&P->d_pull_words, pull_words);
        up(&P->d_slot_ptr, slot_ptr);
        up(&P->d_med, med);
        up(&P->d_med_lits, med_lits);
        up(&P->d_med_slots, med_slots);
        up(&P->d_long, lng);
        up(&P->d_long_lits, long_lits);
        up(&P->d_long_slots, long_slots);
        up(&P->d_count, cnt);
        up(&P->d_count_lits, cnt_lits);
        if (st != AFS_OK) { afs_problem_destroy(P); return st; }
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
    cudaSetDevice(p->device);
    cudaDeviceSynchronize();
    cudaFree(p->d_pull_ptr); cudaFree(p->d_pull_words); cudaFree(p->d_slot_ptr);
    cudaFree(p->d_med); cudaFree(p->d_med_lits); cudaFree(p->d_med_slots);
    cudaFree(p->d_long); cudaFree(p->d_long_lits); cudaFree(p->d_long_slots);
    cudaFree(p->d_count); cudaFree(p->d_count_lits);
    afs::free_workspace(p);
    (void)cudaGetLastError();
    delete p;
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
    case 5: return p->n_long;
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
