// api.cpp - the C ABI of include/kripke.h: argument checking, program staging (H1), class tables
// (H2), kernel selection and launch sequencing.  All compute runs in the CUDA kernels of this
// library; there is no CPU evaluation path here.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <tuple>

#include <chrono>
#include <string>

#include "internal.h"
#include "jit.h"

using namespace kripke;

namespace {

thread_local int g_last_cuda_error = 0;

int cuda_fail(int e) {
    g_last_cuda_error = e;
    return KRIPKE_ECUDA;
}
#define CU(call)                                          \
    do {                                                  \
        cudaError_t e_ = (call);                          \
        if (e_ != cudaSuccess) return cuda_fail((int)e_); \
    } while (0)

template <typename T>
int upload(T **dst, const std::vector<T> &src) {
    *dst = nullptr;
    if (src.empty()) return KRIPKE_OK;
    CU(cudaMalloc((void **)dst, src.size() * sizeof(T)));
    CU(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    return KRIPKE_OK;
}

// A lowered set of records for the sliced kernel plus the list of records it cannot run.  Slots are
// sorted by the number of register-stack slots they need, so that each need class can run on the
// kernel instantiation with the fewest slots (more words per thread, more resident warps).
struct HostPlan {
    std::vector<uint16_t> ucode;
    std::vector<uint32_t> slot_record;
    std::vector<uint32_t> unfit;
    uint32_t stride = 2;
    uint32_t need_end[UC_DMAX + 1] = {0, 0, 0, 0, 0};   // slots with need <= d are [0, need_end[d])
    uint64_t n_modal = 0, n_bool = 0;
};

// skip (may be null): records that are not scanned at all (their program is another record's)
void build_plan(const std::vector<Lowered> &low, const std::vector<bool> &fits, HostPlan *hp,
                const std::vector<bool> *skip = nullptr) {
    auto skipped = [&](size_t i) { return skip && (*skip)[i]; };
    size_t longest = 1;
    for (size_t i = 0; i < low.size(); ++i)
        if (fits[i] && !skipped(i)) longest = std::max(longest, low[i].ucode.size());
    hp->stride = (uint32_t)((longest + 1 + 1) / 2 * 2);        // one spare entry after FIN (prefetch)
    for (size_t i = 0; i < low.size(); ++i)
        if (!fits[i] && !skipped(i)) hp->unfit.push_back((uint32_t)i);
    for (int need = 1; need <= UC_DMAX; ++need) {
        for (size_t i = 0; i < low.size(); ++i) {
            if (!fits[i] || skipped(i) || low[i].need != need) continue;
            hp->slot_record.push_back((uint32_t)i);
            size_t at = hp->ucode.size();
            hp->ucode.resize(at + hp->stride, (uint16_t)UC_FIN_ALL);
            std::memcpy(&hp->ucode[at], low[i].ucode.data(), low[i].ucode.size() * sizeof(uint16_t));
            hp->n_modal += low[i].n_modal;
            hp->n_bool += low[i].n_bool;
        }
        hp->need_end[need] = (uint32_t)hp->slot_record.size();
    }
}

struct DevicePlan {
    uint16_t *ucode = nullptr;
    uint32_t *slot_record = nullptr;
    uint32_t *unfit = nullptr;
    uint32_t *alias = nullptr;         // frame-list plans: (record, representative) pairs of records not scanned themselves
    uint32_t n_slots = 0, n_unfit = 0, stride = 2, n_alias = 0;
    uint32_t need_end[UC_DMAX + 1] = {0, 0, 0, 0, 0};
    uint64_t n_modal = 0, n_bool = 0;
    void release() {
        cudaFree(ucode); cudaFree(slot_record); cudaFree(unfit); cudaFree(alias);
        ucode = nullptr; slot_record = nullptr; unfit = nullptr; alias = nullptr; n_slots = n_unfit = n_alias = 0;
    }
};

int upload_plan(const HostPlan &hp, DevicePlan *dp) {
    dp->release();
    int rc;
    if ((rc = upload(&dp->ucode, hp.ucode)) || (rc = upload(&dp->slot_record, hp.slot_record)) ||
        (rc = upload(&dp->unfit, hp.unfit)))
        return rc;
    dp->n_slots = (uint32_t)hp.slot_record.size();
    dp->n_unfit = (uint32_t)hp.unfit.size();
    dp->stride = hp.stride;
    std::memcpy(dp->need_end, hp.need_end, sizeof(dp->need_end));
    dp->n_modal = hp.n_modal;
    dp->n_bool = hp.n_bool;
    return KRIPKE_OK;
}

// The records of one scan grouped by the number of variables their programs mention (after
// constant folding).  A program that ignores a variable has the same truth set for every value of
// it, so group g is scanned over the 2^(g*n) valuations of its own variables only - Algorithm 1's
// per-formula k_b - and its model count is multiplied by 2^((k-g)*n) (reading R8).
struct GroupPlan {
    uint32_t k_eff = 0;
    DevicePlan dp;                    // every record of the group, for the interpreted bit-sliced / scalar kernels
    bool use_jit = false;             // the group runs on compiled kernels (jit.h) instead of dp
    JitGroupPlan jit;
    uint32_t *d_alias = nullptr;      // device: (record, representative) pairs - records whose lowered program
    uint32_t n_alias = 0;             // equals the representative's are not scanned, they copy its accumulators
    void release() {
        dp.release();
        jit.release();
        cudaFree(d_alias);
        d_alias = nullptr; n_alias = 0;
    }
};
struct ScanPlan {
    std::vector<GroupPlan> groups;
    double jit_compile_seconds = 0.0; // host time spent emitting + compiling + loading (0 if cached or interpreted)
    void release() {
        for (auto &g : groups) g.release();
        groups.clear();
    }
};

// ---- class tables (step H2) ----------------------------------------------------------------------
// Ascending K-indices of the preorders (S4) / equivalences (S5) on n worlds.  Rows are chosen from
// world n-1 (most significant bits of f) down to world 0, each ascending, so the enumeration is
// already in ascending f; a branch is cut as soon as two fixed rows break transitivity / symmetry.
struct TableBuilder {
    uint32_t n, cls;
    uint32_t succ[KRIPKE_MAX_WORLDS];
    std::vector<uint64_t> *out;
    bool fixed_ok(int lo) const {       // rows lo..n-1 are fixed
        for (uint32_t w = lo; w < n; ++w)
            for (uint32_t u = lo; u < n; ++u) {
                if (((succ[w] >> u) & 1u) && (succ[u] & ~succ[w])) {
                    // u in succ[w] needs succ[u] subset of succ[w]; only bits of fixed rows are final,
                    // but succ[] rows are complete masks, so the test is exact for fixed w, u
                    return false;
                }
                if (cls == KRIPKE_CLASS_S5 && (((succ[w] >> u) & 1u) != ((succ[u] >> w) & 1u))) return false;
            }
        return true;
    }
    void rec(int w) {
        if (w < 0) {
            uint64_t f = 0;
            for (uint32_t x = 0; x < n; ++x) f |= (uint64_t)succ[x] << (x * n);
            out->push_back(f);
            return;
        }
        for (uint32_t m = 0; m < (1u << n); ++m) {
            if (!((m >> w) & 1u)) continue;     // reflexive
            succ[w] = m;
            if (fixed_ok(w)) rec(w - 1);
        }
    }
};

std::mutex g_table_mutex;
std::map<std::pair<uint32_t, uint32_t>, std::vector<uint64_t>> g_tables_host;
std::map<std::tuple<int, uint32_t, uint32_t>, uint64_t *> g_tables_dev;

}  // namespace

namespace kripke {

// For entry points that live in other translation units (scan_static.cu): record a cudaError_t where
// kripke_last_cuda_error() finds it and return KRIPKE_ECUDA.
int note_cuda_error(int e) { return cuda_fail(e); }

const std::vector<uint64_t> *class_table_host(uint32_t n, uint32_t cls) {
    std::lock_guard<std::mutex> lock(g_table_mutex);
    auto key = std::make_pair(n, cls);
    auto it = g_tables_host.find(key);
    if (it == g_tables_host.end()) {
        std::vector<uint64_t> v;
        TableBuilder tb;
        tb.n = n; tb.cls = cls; tb.out = &v;
        std::memset(tb.succ, 0, sizeof(tb.succ));
        tb.rec((int)n - 1);
        it = g_tables_host.emplace(key, std::move(v)).first;
    }
    return &it->second;
}

}  // namespace kripke

namespace {

int class_table_device(uint32_t n, uint32_t cls, const uint64_t **out) {
    *out = nullptr;
    if (cls != KRIPKE_CLASS_S4 && cls != KRIPKE_CLASS_S5) return KRIPKE_OK;
    int dev = 0;
    CU(cudaGetDevice(&dev));
    const std::vector<uint64_t> *h = class_table_host(n, cls);
    std::lock_guard<std::mutex> lock(g_table_mutex);
    auto key = std::make_tuple(dev, n, cls);
    auto it = g_tables_dev.find(key);
    if (it == g_tables_dev.end()) {
        uint64_t *d = nullptr;
        int rc = upload(&d, *h);
        if (rc) return rc;
        it = g_tables_dev.emplace(key, d).first;
    }
    *out = it->second;
    return KRIPKE_OK;
}

int class_size(uint32_t n, uint32_t cls, uint64_t *out) {
    if (n < 1 || n > KRIPKE_MAX_WORLDS || cls > KRIPKE_CLASS_S5) return KRIPKE_EINVAL;
    if (cls == KRIPKE_CLASS_K) *out = 1ull << (n * n);
    else if (cls == KRIPKE_CLASS_T) *out = 1ull << (n * n - n);
    else *out = class_table_host(n, cls)->size();
    return KRIPKE_OK;
}

}  // namespace

struct kripke_programs {
    uint32_t n_formulas = 0, n_vars = 0;
    std::vector<uint8_t> h_code;
    std::vector<uint32_t> h_offsets;
    uint8_t *d_code = nullptr;
    uint32_t *d_offsets = nullptr;
    // per formula, from the postfix program as written: modal operators, binary connectives, variables
    std::vector<uint32_t> f_modal, f_binary, f_vars;
    std::map<uint64_t, ScanPlan> single;     // one record per formula; cached per (n, k, class, flags, engine)
    std::map<uint64_t, ScanPlan> density;    // failure-density plans, per (n, k, class)
    struct PairPlan {                  // plans of kripke_distinguish_pairs, cached per pair list and shape
        std::vector<uint32_t> pairs;
        uint64_t key = 0;
        ScanPlan plan;
        uint32_t *d_pairs = nullptr;
        uint64_t last_use = 0;
    };
    std::vector<PairPlan *> pair_plans;
    uint64_t use_clock = 0;
    cudaEvent_t done = nullptr;        // end of the last scan enqueued on this handle
    void *last_stream = nullptr;
    bool has_last = false;
    bool aux_work = false;             // something other than a scan (bitmaps, densities, signatures, the size loop's
                                       // record kernel) was enqueued on this handle's memory: not covered by `done`
    DevicePlan list_single;            // frame-list mode: every formula lowered without derived leaves
    bool list_single_built = false;
    DevicePlan list_pair;              // plan of the last pair list given to kripke_distinguish_pairs_frames
    std::vector<uint32_t> list_pair_key;   // that list (a call with the same list reuses the plan and enqueues only)
    bool list_pair_built = false;
    uint32_t *d_pairs = nullptr;
    uint32_t pairs_cap = 0;
    Accum *d_accum = nullptr;
    uint32_t accum_cap = 0;
    kripke_count_t *d_tmp_counts = nullptr;   // per-layer scratch of the size loop
    kripke_witness_t *d_tmp_wit = nullptr;
    uint32_t tmp_cap = 0;
    kripke_run_info_t last = {};
};

namespace {

int ensure_accum(kripke_programs *h, uint32_t n) {
    if (n <= h->accum_cap) return KRIPKE_OK;
    cudaFree(h->d_accum);
    h->d_accum = nullptr; h->accum_cap = 0;
    CU(cudaMalloc((void **)&h->d_accum, (size_t)n * sizeof(Accum)));
    h->accum_cap = n;
    return KRIPKE_OK;
}

// Which reduced shapes (n, g), g < k, the sliced kernel can run for this class: bit g.
// Bit 31 says "class other than K": such scans can only use the frame-per-unit instantiations, whose
// lowering mode differs (sliced_lower_mode), so their plans are built and cached separately.
constexpr uint32_t SHAPES_NOT_K = 1u << 31;
constexpr uint32_t SHAPES_NO_SHARING = 1u << 30;      // KRIPKE_NO_SHARING: scan every record itself
uint32_t reduced_shapes(uint32_t n, uint32_t k, uint32_t cls, uint32_t flags) {
    uint32_t mask = (cls != KRIPKE_CLASS_K ? SHAPES_NOT_K : 0u) | ((flags & KRIPKE_NO_SHARING) ? SHAPES_NO_SHARING : 0u);
    if ((flags & KRIPKE_FULL_SWEEP) || (flags & KRIPKE_KERNEL_MASK) == KRIPKE_KERNEL_SCALAR) return mask;
    if (n < 1 || n > KRIPKE_MAX_WORLDS || k > KRIPKE_MAX_VARS) return mask;
    if (!sliced_select(n, k, cls, 1, nullptr)) return mask;
    for (uint32_t g = 0; g < k; ++g)
        if (sliced_select(n, g, cls, 1, nullptr)) mask |= 1u << g;
    return mask;
}

// Engines of a scan plan.
enum : uint32_t { ENGINE_INTERPRETED = 0, ENGINE_JIT = 1 };

// Tunables of the compiled scans (kripke_jit_configure).
uint32_t g_jit_max_programs = 48;
uint32_t g_jit_min_blocks = 2;

// Lowers the records (formulas, or pairs if `pairs` != null) into one GroupPlan per variable count.
int build_scan_plan(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                    uint32_t shapes, ScanPlan *out);
int build_jit_plan(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                   uint32_t cls, uint32_t flags, ScanPlan *out);

constexpr uint32_t SCAN_FLAGS = KRIPKE_ACCUMULATE | KRIPKE_FULL_SWEEP | KRIPKE_NO_SHARING | KRIPKE_NO_SUBTERM_SHARING |
                                KRIPKE_NO_GUARDED_ROOTS | KRIPKE_NO_BOX_DISTRIBUTION |
                                KRIPKE_KERNEL_MASK | KRIPKE_REDUCE_MASK;

// Argument checks of every class scan - before any plan is built or cached.
int check_scan_args(const kripke_programs *h, uint32_t n_records, uint32_t n, uint32_t k, uint32_t cls, uint64_t begin,
                    uint64_t count, uint32_t flags, const void *counts_out, const void *witness_out) {
    if (n < 1 || n > KRIPKE_MAX_WORLDS || k != h->n_vars || cls > KRIPKE_CLASS_S5) return KRIPKE_EINVAL;
    if (n * n + k * n > KRIPKE_MAX_MODEL_BITS) return KRIPKE_EUNSUPPORTED;
    if (flags & ~SCAN_FLAGS) return KRIPKE_EINVAL;
    if (((flags & KRIPKE_REDUCE_MASK) >> 8) > 2) return KRIPKE_EINVAL;
    if (n_records && (!counts_out || !witness_out)) return KRIPKE_EINVAL;
    uint64_t csize = 0;
    int rc = class_size(n, cls, &csize);
    if (rc) return rc;
    if (begin > csize || count > csize - begin) return KRIPKE_EINVAL;
    return KRIPKE_OK;
}

// Which engine a scan with these flags uses: compiled kernels whenever the emitter has a layout for
// the full shape (AUTO) or when forced; the interpreted kernels otherwise.
int pick_engine(uint32_t n, uint32_t k, uint32_t cls, uint32_t flags, uint32_t *engine) {
    const uint32_t family = flags & KRIPKE_KERNEL_MASK;
    const bool can = jit_layout(n, k, cls, nullptr);
    if (family == KRIPKE_KERNEL_JIT && !can) return KRIPKE_EUNSUPPORTED;
    *engine = (can && (family == KRIPKE_KERNEL_JIT || family == KRIPKE_KERNEL_AUTO)) ? ENGINE_JIT : ENGINE_INTERPRETED;
    return KRIPKE_OK;
}

// The common scan: zero accumulators, run every group on the compiled or interpreted bit-sliced kernels
// where they apply (aligned part of the range) and on the scalar kernel elsewhere, then finish.
int run_scan(kripke_programs *h, const ScanPlan &plan, const uint32_t *h_pairs, const uint32_t *d_pairs, uint32_t n_records,
             uint32_t n, uint32_t k, uint32_t cls, uint64_t begin, uint64_t count, uint32_t flags,
             kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream) {
    int rc = check_scan_args(h, n_records, n, k, cls, begin, count, flags, counts_out, witness_out);
    if (rc) return rc;
    const uint32_t family = flags & KRIPKE_KERNEL_MASK, reduce = (flags & KRIPKE_REDUCE_MASK) >> 8;
    h->last = kripke_run_info_t{};
    h->last.models_per_program = count << (k * n);
    h->last.jit_compile_seconds = plan.jit_compile_seconds;
    // SURVEY 8(d)'s algorithmic operation count, per FORMULA of the batch as written (no sharing, no folding):
    // (d n^2 + b n + n + 1) 3-input logic instructions per 32-model word, 2^(k_b n) / 32 words per frame
    {
        auto alg = [&](uint32_t f, uint32_t kb) {
            return (double)(h->f_modal[f] * n * n + h->f_binary[f] * n) * (double)(1ull << (kb * n)) / 32.0;
        };
        auto nv = [](uint32_t m) { uint32_t c = 0; for (; m; m >>= 1) c += m & 1u; return c; };
        for (uint32_t r = 0; r < n_records; ++r) {
            if (h_pairs) {
                const uint32_t fa = h_pairs[2 * r], fb = h_pairs[2 * r + 1], kb = nv(h->f_vars[fa] | h->f_vars[fb]);
                h->last.algorithmic_logic_instr_per_frame += alg(fa, kb) + alg(fb, kb) + (double)(2 * n + 1) * (double)(1ull << (kb * n)) / 32.0;
            } else {
                const uint32_t kb = nv(h->f_vars[r]);
                h->last.algorithmic_logic_instr_per_frame += alg(r, kb) + (double)(n + 1) * (double)(1ull << (kb * n)) / 32.0;
            }
        }
    }
    for (size_t gi = 0; gi < plan.groups.size(); ++gi) {
        const GroupPlan &g = plan.groups[gi];
        // bookkeeping for the roofline: instructions the kernels need per frame of the range
        const double words = (double)(1ull << (g.k_eff * n)) / 32.0;
        if (g.use_jit) {
            h->last.sliced_logic_ops_per_word += g.jit.stats.logic_ops_emitted;
            h->last.logic_instr_per_frame += g.jit.stats.logic_ops_per_word * words;
            h->last.popc_instr_per_frame += (double)g.jit.n_slots * words;
            h->last.executed_models += (uint64_t)g.jit.n_slots * (count << (g.k_eff * n));
            h->last.jit_programs += g.jit.n_slots;
            continue;
        }
        auto dense = [&](const DevicePlan &dp) {
            return (double)(dp.n_modal * n * n + dp.n_bool * n + (uint64_t)dp.n_slots * (n + 1)) * words;
        };
        h->last.sliced_logic_ops_per_word += g.dp.n_modal * n * n + g.dp.n_bool * n + (uint64_t)g.dp.n_slots * (n + 1);
        h->last.logic_instr_per_frame += dense(g.dp);
        h->last.popc_instr_per_frame += (double)g.dp.n_slots * words;
        h->last.executed_models += (uint64_t)(g.dp.n_slots + g.dp.n_unfit) * (count << (g.k_eff * n));
    }
    if (n_records == 0) return KRIPKE_OK;

    // One scan at a time per handle (its accumulators are shared): a call on another stream waits for
    // the previous call's work on the device, it never blocks the host.
    if (!h->done) CU(cudaEventCreateWithFlags(&h->done, cudaEventDisableTiming));
    if (h->has_last && h->last_stream != stream) CU(cudaStreamWaitEvent((cudaStream_t)stream, h->done, 0));
    if (n_records > h->accum_cap && h->has_last) CU(cudaEventSynchronize(h->done));   // the buffer is about to be replaced
    if ((rc = ensure_accum(h, n_records))) return rc;
    ScanJob job;
    job.n = n; job.k = k; job.cls = cls;
    job.frame_begin = begin; job.frame_count = count;
    if ((rc = class_table_device(n, cls, &job.class_table))) return rc;
    job.code = h->d_code; job.offsets = h->d_offsets; job.n_formulas = h->n_formulas;
    job.pairs = d_pairs; job.n_records = n_records;
    job.accum = h->d_accum;

    // A forced compiled scan needs a unit-aligned range: refused here, before anything is enqueued.
    if (family == KRIPKE_KERNEL_JIT)
        for (const GroupPlan &g : plan.groups)
            if (g.use_jit) {
                const uint64_t fpu = 1ull << g.jit.lay.unit_frames_log2;
                if (begin % fpu || (begin + count) % fpu) return KRIPKE_EUNSUPPORTED;
            }

    int e = launch_init(job.accum, n_records, stream);
    if (e) return cuda_fail(e);
    uint32_t launches = 1;

    // Everything from here on works on the handle's accumulators.  Whatever this call manages to enqueue - also
    // when it then gives up (a forced family that does not fit, a failed launch) - has to be ordered before the
    // next call on the handle, so the enqueueing is one function and the event is recorded on every way out.
    auto enqueue = [&]() -> int {
    if (family == KRIPKE_KERNEL_SCALAR) {
        if ((e = launch_scalar(job, nullptr, n_records, reduce, stream, &launches))) return cuda_fail(e);
    }
    // the records of one group on the bit-sliced kernel where an instantiation exists (aligned part of
    // the range), on the scalar kernel elsewhere
    auto run_sliced_or_scalar = [&](const DevicePlan &dp, uint32_t k_eff) -> int {
        uint32_t max_need = 0;
        for (uint32_t d = 1; d <= (uint32_t)UC_DMAX; ++d)
            if (dp.need_end[d] > dp.need_end[d - 1]) max_need = d;
        uint64_t fpu = 1;
        bool use_sliced = dp.n_slots > 0 && sliced_select(n, k_eff, cls, 1, &fpu);
        uint64_t ab = begin, ae = begin;          // aligned sub-range for the sliced kernel
        if (use_sliced) {
            // the need classes may run on instantiations with different unit sizes (powers of two):
            // align the range to the largest one in use
            for (uint32_t d = 2; d <= (uint32_t)UC_DMAX; ++d) {
                uint64_t f2 = 1;
                if (dp.need_end[d] > dp.need_end[d - 1] && sliced_select(n, k_eff, cls, d, &f2)) fpu = std::max(fpu, f2);
            }
            ab = (begin + fpu - 1) / fpu * fpu;
            ae = (begin + count) / fpu * fpu;
            if (ae <= ab) { use_sliced = false; ab = ae = begin; }
        }
        if (family == KRIPKE_KERNEL_SLICED) {
            if ((dp.n_slots && !use_sliced) || dp.n_unfit || ab != begin || ae != begin + count ||
                (dp.n_slots && !sliced_select(n, k_eff, cls, max_need, nullptr)))
                return KRIPKE_EUNSUPPORTED;
        }
        int e = 0;
        if (use_sliced) {
            ScanJob sj = job;                     // scalar launches on the sub-range (true k)
            sj.frame_begin = ab; sj.frame_count = ae - ab;
            ScanJob rj = sj;                      // the reduced scan: its own variable count
            rj.k = k_eff;
            if (h->last.kernel_family == 0) h->last.kernel_family = 1;
            // consecutive need classes that map to the same instantiation run as one launch
            uint32_t d = 1;
            while (d <= (uint32_t)UC_DMAX) {
                uint32_t lo = dp.need_end[d - 1], hi = dp.need_end[d], top = d;
                const uint32_t row = sliced_row(n, k_eff, cls, d);
                while (top < (uint32_t)UC_DMAX && sliced_row(n, k_eff, cls, top + 1) == row) { ++top; hi = dp.need_end[top]; }
                if (hi > lo) {
                    if (row == UINT32_MAX) {       // no instantiation keeps this many slots: scalar kernel
                        if ((e = launch_scalar(sj, dp.slot_record + lo, hi - lo, reduce, stream, &launches)))
                            return cuda_fail(e);
                    } else {
                        SlicedPlan sp;
                        sp.ucode = dp.ucode + (size_t)lo * dp.stride;
                        sp.slot_record = dp.slot_record + lo;
                        sp.n_slots = hi - lo; sp.stride = dp.stride; sp.max_need = top;
                        sp.model_shift = (k - k_eff) * n;
                        if ((e = launch_sliced(rj, sp, stream, &launches))) return cuda_fail(e);
                    }
                }
                d = top + 1;
            }
            ScanJob head = job, tail = job;
            head.frame_count = ab - begin;
            tail.frame_begin = ae; tail.frame_count = begin + count - ae;
            if ((e = launch_scalar(head, dp.slot_record, dp.n_slots, reduce, stream, &launches))) return cuda_fail(e);
            if ((e = launch_scalar(tail, dp.slot_record, dp.n_slots, reduce, stream, &launches))) return cuda_fail(e);
        } else if (dp.n_slots) {
            if ((e = launch_scalar(job, dp.slot_record, dp.n_slots, reduce, stream, &launches))) return cuda_fail(e);
        }
        if (dp.n_unfit && (e = launch_scalar(job, dp.unfit, dp.n_unfit, reduce, stream, &launches)))
            return cuda_fail(e);
        return KRIPKE_OK;
    };
    for (size_t gi = 0; gi < plan.groups.size(); ++gi) {
        if (family == KRIPKE_KERNEL_SCALAR) break;
        const GroupPlan &g = plan.groups[gi];
        if (!g.use_jit) {
            if ((rc = run_sliced_or_scalar(g.dp, g.k_eff))) return rc;
            continue;
        }
        // compiled kernels on the unit-aligned part of the range, scalar kernel on the ragged ends
        const uint64_t fpu = 1ull << g.jit.lay.unit_frames_log2;
        uint64_t ab = (begin + fpu - 1) / fpu * fpu, ae = (begin + count) / fpu * fpu;
        if (ae <= ab) ab = ae = begin;
        if (family == KRIPKE_KERNEL_JIT && (ab != begin || ae != begin + count)) return KRIPKE_EUNSUPPORTED;
        if (ae > ab) {
            ScanJob rj = job;
            rj.k = g.k_eff; rj.frame_begin = ab; rj.frame_count = ae - ab;
            h->last.kernel_family = 2;
            if ((e = jit_launch_group(rj, g.jit, (k - g.k_eff) * n, nullptr, stream, &launches))) return cuda_fail(e);
        }
        ScanJob head = job, tail = job;
        head.frame_count = ab - begin;
        tail.frame_begin = ae; tail.frame_count = begin + count - ae;
        if ((e = launch_scalar(head, g.jit.d_slot_record, g.jit.n_slots, reduce, stream, &launches))) return cuda_fail(e);
        if ((e = launch_scalar(tail, g.jit.d_slot_record, g.jit.n_slots, reduce, stream, &launches))) return cuda_fail(e);
    }
    // records that share a representative's lowered program take its accumulators (the scalar family
    // scanned every record itself)
    if (family != KRIPKE_KERNEL_SCALAR)
        for (const GroupPlan &g : plan.groups)
            if (g.n_alias) {
                if ((e = launch_alias_accum(job.accum, g.d_alias, g.n_alias, stream))) return cuda_fail(e);
                ++launches;
            }
    if ((e = launch_finish(job, (flags & KRIPKE_ACCUMULATE) != 0, counts_out, witness_out, stream)))
        return cuda_fail(e);
    return KRIPKE_OK;
    };
    rc = enqueue();
    const cudaError_t recorded = cudaEventRecord(h->done, (cudaStream_t)stream);
    h->last_stream = stream;
    h->has_last = true;
    if (rc) return rc;
    if (recorded != cudaSuccess) return cuda_fail((int)recorded);
    h->last.launches = launches + 1;
    return KRIPKE_OK;
}

int build_scan_plan(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                    uint32_t shapes, ScanPlan *out) {
    out->release();
    auto prog = [&](uint32_t f) { return &h->h_code[h->h_offsets[f]]; };
    auto plen = [&](uint32_t f) { return h->h_offsets[f + 1] - h->h_offsets[f]; };
    // group of every record: the least usable variable count that covers its support
    std::vector<uint32_t> support(n_records), group(n_records);
    for (uint32_t r = 0; r < n_records; ++r) {
        uint32_t s = pairs ? (program_support(prog(pairs[2 * r]), plen(pairs[2 * r])) |
                              program_support(prog(pairs[2 * r + 1]), plen(pairs[2 * r + 1])))
                           : program_support(prog(r), plen(r));
        support[r] = s;
        uint32_t cnt = 0;
        for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) cnt += (s >> i) & 1u;
        uint32_t g = cnt;
        while (g < k && !((shapes >> g) & 1u)) ++g;
        group[r] = g;
    }
    for (uint32_t g = 0; g <= k; ++g) {
        std::vector<uint32_t> recs;
        for (uint32_t r = 0; r < n_records; ++r)
            if (group[r] == g) recs.push_back(r);
        if (recs.empty()) continue;
        const uint32_t mode = sliced_lower_mode(n, g, (shapes & SHAPES_NOT_K) ? KRIPKE_CLASS_T : KRIPKE_CLASS_K);
        std::vector<Lowered> low(recs.size());
        std::vector<bool> fits(recs.size());
        for (size_t i = 0; i < recs.size(); ++i) {
            const uint32_t r = recs[i];
            uint8_t rename[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
            uint8_t next = 0;
            for (uint32_t v = 0; v < KRIPKE_MAX_VARS; ++v)
                if ((support[r] >> v) & 1u) rename[v] = next++;
            if (g == k) for (uint32_t v = 0; v < KRIPKE_MAX_VARS; ++v) rename[v] = (uint8_t)v;   // full sweep: as written
            auto lower = [&](uint32_t m) {
                return pairs ? lower_pair(prog(pairs[2 * r]), plen(pairs[2 * r]), prog(pairs[2 * r + 1]),
                                          plen(pairs[2 * r + 1]), m, rename, &low[i])
                             : lower_single(prog(r), plen(r), m, rename, &low[i]);
            };
            auto lower_for_kernel = [&]() {
                bool ok = lower(mode);
                if (ok && (mode & LOWER_FUSE) && !sliced_fuses(n, g, (uint32_t)low[i].need)) {
                    low[i] = Lowered();
                    ok = lower(mode & ~(uint32_t)LOWER_FUSE);
                }
                return ok;
            };
            fits[i] = lower_for_kernel();
            // Counts and the least refuting frame do not depend on which variable plays which role (a
            // permutation of the variables permutes the valuations of every frame), so with sharing on
            // the cheapest - then lexicographically least - of the permuted lowerings is taken: more
            // programs coincide, and the in-word variable p_0 lands where it saves most.
            if (g >= 2 && !(shapes & SHAPES_NO_SHARING)) {
                uint8_t perm[KRIPKE_MAX_VARS] = {0, 1, 2, 3}, base[KRIPKE_MAX_VARS];
                std::copy(rename, rename + KRIPKE_MAX_VARS, base);
                auto cost = [&](const Lowered &l) { return (uint64_t)l.n_modal * n * n + (uint64_t)l.n_bool * n; };
                Lowered best = low[i];
                bool best_ok = fits[i];
                while (std::next_permutation(perm, perm + g)) {
                    for (uint32_t v = 0; v < KRIPKE_MAX_VARS; ++v) rename[v] = base[v] < g ? perm[base[v]] : base[v];
                    low[i] = Lowered();
                    const bool ok = lower_for_kernel();
                    if (!ok) continue;
                    if (!best_ok || cost(low[i]) < cost(best) ||
                        (cost(low[i]) == cost(best) && (low[i].need < best.need ||
                                                        (low[i].need == best.need && low[i].ucode < best.ucode)))) {
                        best = low[i];
                        best_ok = true;
                    }
                }
                low[i] = best;
                fits[i] = best_ok;
            }
        }
        // Records of the group whose lowered programs are identical (alpha-equivalent after the variable
        // renaming, or equal after constant folding) are scanned once: the first is the representative,
        // the others receive a copy of its accumulators before the finish step (DESIGN.md 5.1 "Sharing").
        std::vector<uint32_t> alias;
        if (!(shapes & SHAPES_NO_SHARING)) {
            std::map<std::vector<uint16_t>, uint32_t> seen;
            std::vector<uint32_t> recs2;
            std::vector<Lowered> low2;
            std::vector<bool> fits2;
            for (size_t i = 0; i < recs.size(); ++i) {
                if (fits[i]) {
                    auto it = seen.find(low[i].ucode);
                    if (it != seen.end()) { alias.push_back(recs[i]); alias.push_back(it->second); continue; }
                    seen.emplace(low[i].ucode, recs[i]);
                }
                recs2.push_back(recs[i]);
                low2.push_back(std::move(low[i]));
                fits2.push_back(fits[i]);
            }
            recs.swap(recs2); low.swap(low2); fits.swap(fits2);
        }
        HostPlan hp;
        build_plan(low, fits, &hp);
        for (auto &x : hp.slot_record) x = recs[x];       // slot -> record index of the whole batch
        for (auto &x : hp.unfit) x = recs[x];
        GroupPlan gp;
        gp.k_eff = g;
        int rc = upload_plan(hp, &gp.dp);
        if (!rc) rc = upload(&gp.d_alias, alias);
        if (rc) { gp.release(); out->release(); return rc; }
        gp.n_alias = (uint32_t)(alias.size() / 2);
        out->groups.push_back(gp);
    }
    return KRIPKE_OK;
}

// ---- compiled scans (jit.h) -----------------------------------------------------------------------
// The records of one variable-count group as roots of one graph.  Host only.
struct JitGroupHost {
    uint32_t g = 0;
    Dag dag;
    std::vector<JitRoot> roots;          // distinct roots = the programs that are scanned
    std::vector<uint32_t> slot_record;   // representative record of each root
    std::vector<uint32_t> alias;         // (record, representative) pairs
    JitOptStats opt;
};

// Where a record went, and the variable order it is evaluated under (host checks only).
struct JitRecordInfo {
    uint32_t group = 0, slot = 0, support = 0, neg = 0;
    uint8_t rename[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
};

// Groups the records by the number of variables they mention (Algorithm 1's per-formula k_b; the
// least g >= that count for which the emitter has a layout) and builds each group's graph.
int jit_group_records(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                      uint32_t cls, uint32_t flags, uint32_t mode, std::vector<JitGroupHost> *out,
                      std::vector<JitRecordInfo> *info_out = nullptr) {
    auto layout_ok = [&](uint32_t g) {
        return mode == JIT_MODE_DENSITY ? jit_density_layout(n, g, cls, nullptr) : jit_layout(n, g, cls, nullptr);
    };
    auto prog = [&](uint32_t f) { return &h->h_code[h->h_offsets[f]]; };
    auto plen = [&](uint32_t f) { return h->h_offsets[f + 1] - h->h_offsets[f]; };
    out->clear();
    out->resize(k + 1);
    for (uint32_t g = 0; g <= k; ++g) (*out)[g].g = g;
    std::vector<Dag> probe(k + 1);       // unsalted graphs: which records are the same program
    // per group: which of its variables change inside a thread's word loop on the group's layout
    std::vector<uint32_t> loop_vars(k + 1, 0);
    for (uint32_t g = 0; g <= k; ++g) {
        JitLayout lay;
        if (!(mode == JIT_MODE_DENSITY ? jit_density_layout(n, g, cls, &lay) : jit_layout(n, g, cls, &lay))) continue;
        for (uint32_t v = 0; v < g; ++v)
            for (uint32_t w = 0; w < n; ++w)
                if (jit_atom_level(lay, v, w) > 0) loop_vars[g] |= 1u << v;
    }
    std::vector<std::map<std::pair<uint32_t, uint32_t>, uint32_t>> seen(k + 1);
    if (info_out) info_out->assign(n_records, JitRecordInfo());
    for (uint32_t r = 0; r < n_records; ++r) {
        const uint32_t fa = pairs ? pairs[2 * r] : r, fb = pairs ? pairs[2 * r + 1] : r;
        // the variables the record's GRAPH mentions (the rewrites fold more than the syntax shows: x & ~x, box T)
        uint32_t sup;
        {
            Dag sd;
            sup = sd.support(sd.build(prog(fa), plen(fa), nullptr));
            if (pairs) sup |= sd.support(sd.build(prog(fb), plen(fb), nullptr));
        }
        uint32_t cnt = 0;
        for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) cnt += (sup >> i) & 1u;
        uint32_t g = (flags & KRIPKE_FULL_SWEEP) ? k : cnt;
        while (g < k && !layout_ok(g)) ++g;
        if (!layout_ok(g)) return KRIPKE_EUNSUPPORTED;
        JitGroupHost &G = (*out)[g];
        uint8_t rename[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
        uint32_t neg = 0;
        if (flags & KRIPKE_NO_SHARING) {                 // variables in their own order, nothing shared
            uint8_t next = 0;
            for (uint32_t v = 0; v < KRIPKE_MAX_VARS; ++v)
                if ((sup >> v) & 1u) rename[v] = next++;
        } else {
            canonical_rename(prog(fa), plen(fa), pairs ? prog(fb) : nullptr, pairs ? plen(fb) : 0u, sup, n, loop_vars[g], rename, &neg);
        }
        if (info_out) {
            JitRecordInfo &ri = (*info_out)[r];
            ri.group = g;
            ri.support = sup;
            ri.neg = neg;
            for (uint32_t v = 0; v < KRIPKE_MAX_VARS; ++v) ri.rename[v] = rename[v];
            ri.slot = (uint32_t)G.roots.size();
        }
        if (!(flags & KRIPKE_NO_SHARING)) {
            // records whose graphs coincide are scanned once (the pair path is symmetric in its two formulas;
            // density mode: the program writes the rows of all its records)
            uint32_t pa = probe[g].build(prog(fa), plen(fa), rename, neg);
            uint32_t pb = pairs ? probe[g].build(prog(fb), plen(fb), rename, neg) : UINT32_MAX;
            if (pairs && pb < pa) std::swap(pa, pb);
            auto it = seen[g].find(std::make_pair(pa, pb));
            if (it != seen[g].end()) {
                G.alias.push_back(r); G.alias.push_back(it->second);
                if (info_out) (*info_out)[r].slot = (*info_out)[it->second].slot;
                continue;
            }
            seen[g].emplace(std::make_pair(pa, pb), r);
        }
        G.dag.salt = (flags & (KRIPKE_NO_SHARING | KRIPKE_NO_SUBTERM_SHARING)) ? r + 1 : 0u;
        JitRoot root;
        root.a = G.dag.build(prog(fa), plen(fa), rename, neg);
        root.b = pairs ? G.dag.build(prog(fb), plen(fb), rename, neg) : UINT32_MAX;
        G.roots.push_back(root);
        G.slot_record.push_back(r);
    }
    // evaluation forms (jit.h): the refutation test pushed through the top of each formula, then box
    // redistributed over conjunctions where the batch makes that cheaper
    for (JitGroupHost &G : *out) {
        if (G.roots.empty()) continue;
        JitLayout lay;
        if (!(mode == JIT_MODE_DENSITY ? jit_density_layout(n, G.g, cls, &lay) : jit_layout(n, G.g, cls, &lay))) continue;
        // (with no variables the frame bits are the lanes and the word loop: the guard sets of class K would be
        // recomputed per word)
        if (mode == JIT_MODE_SCAN && !pairs && !(flags & KRIPKE_NO_GUARDED_ROOTS) && (lay.kn >= 5 || cls != KRIPKE_CLASS_K))
            jit_guard_roots(G.dag, &G.roots);
        if (!(flags & (KRIPKE_NO_SHARING | KRIPKE_NO_SUBTERM_SHARING | KRIPKE_NO_BOX_DISTRIBUTION))) {
            Dag opt;
            jit_optimize(G.dag, lay, &G.roots, &opt, &G.opt);
            G.dag = std::move(opt);
        }
    }
    return KRIPKE_OK;
}

// Process-wide cache of compiled plans, keyed by everything a plan depends on (the programs' bytes, the record
// list, shape, class, flags, emitter configuration) and compared in full: the same batch staged again - a new
// handle for the next class range, shard or call of kripke_eval_batch_host - skips graph building, rewriting,
// emission and compilation and only uploads its slot tables.  The kernels themselves live in the module cache of
// jit_runtime.cpp and are never unloaded.
struct CachedJitGroup {
    uint32_t g = 0;
    JitGroupPlan jit;                 // d_slot_record is null here
    std::vector<uint32_t> alias;
};
struct CachedJitPlan {
    std::vector<CachedJitGroup> groups;
    uint64_t stamp = 0;
};
std::mutex g_plan_cache_mutex;
std::map<std::string, CachedJitPlan> g_plan_cache;
std::atomic<int> g_live_handles{0};            // kripke_programs_t objects alive (their plans hold kernel handles)
uint64_t g_plan_cache_clock = 0;
constexpr size_t PLAN_CACHE_ENTRIES = 32;

std::string jit_plan_key(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                         uint32_t cls, uint32_t flags, uint32_t mode) {
    int dev = 0;
    cudaGetDevice(&dev);
    const uint32_t head[] = {n_records, n, k, cls, flags, mode, g_jit_max_programs, g_jit_min_blocks, (uint32_t)dev,
                             h->n_formulas, pairs ? 1u : 0u};
    std::string key((const char *)head, sizeof(head));
    key.append((const char *)h->h_offsets.data(), h->h_offsets.size() * sizeof(uint32_t));
    key.append((const char *)h->h_code.data(), h->h_code.size());
    if (pairs) key.append((const char *)pairs, 2 * (size_t)n_records * sizeof(uint32_t));
    return key;
}

// Instantiates a cached plan for this handle (device copies of the slot and alias tables).
int instantiate_jit_plan(const CachedJitPlan &cp, ScanPlan *out) {
    for (const CachedJitGroup &cg : cp.groups) {
        GroupPlan gp;
        gp.k_eff = cg.g;
        gp.use_jit = true;
        gp.jit = cg.jit;
        gp.jit.d_slot_record = gp.jit.d_row_begin = gp.jit.d_rows = nullptr;
        int rc = jit_upload_slots(&gp.jit);
        if (rc > 0) rc = cuda_fail(rc);
        if (!rc) rc = upload(&gp.d_alias, cg.alias);
        if (rc) { gp.release(); out->release(); return rc; }
        gp.n_alias = (uint32_t)(cg.alias.size() / 2);
        out->groups.push_back(gp);
    }
    return KRIPKE_OK;
}

int build_jit_plan_mode(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                        uint32_t cls, uint32_t flags, uint32_t mode, ScanPlan *out) {
    out->release();
    const auto t0 = std::chrono::steady_clock::now();
    const uint32_t plan_flags = flags & (KRIPKE_FULL_SWEEP | KRIPKE_NO_SHARING | KRIPKE_NO_SUBTERM_SHARING |
                                         KRIPKE_NO_GUARDED_ROOTS | KRIPKE_NO_BOX_DISTRIBUTION);
    const std::string key = jit_plan_key(h, pairs, n_records, n, k, cls, plan_flags, mode);
    {
        std::lock_guard<std::mutex> lock(g_plan_cache_mutex);
        auto it = g_plan_cache.find(key);
        if (it != g_plan_cache.end()) {
            it->second.stamp = ++g_plan_cache_clock;
            return instantiate_jit_plan(it->second, out);          // jit_compile_seconds stays 0: nothing was compiled
        }
    }
    std::vector<JitGroupHost> groups;
    int rc = jit_group_records(h, pairs, n_records, n, k, cls, flags, mode, &groups);
    if (rc) return rc;
    CachedJitPlan cp;
    for (JitGroupHost &G : groups) {
        if (G.roots.empty() && G.alias.empty()) continue;
        CachedJitGroup cg;
        cg.g = G.g;
        cg.alias = G.alias;
        JitLayout lay;
        if (mode == JIT_MODE_DENSITY) jit_density_layout(n, G.g, cls, &lay);
        else jit_layout(n, G.g, cls, &lay);
        std::string log;
        // density: fewer programs per kernel than a scan - every program keeps n failing-world words alive for its stores
        const uint32_t max_programs = mode == JIT_MODE_DENSITY ? std::min<uint32_t>(g_jit_max_programs, 32) : g_jit_max_programs;
        rc = jit_build_group(G.dag, lay, G.roots, G.slot_record, max_programs, g_jit_min_blocks, mode, &cg.jit, &log);
        cudaFree(cg.jit.d_slot_record);                             // the cache keeps host data only
        cg.jit.d_slot_record = nullptr;
        if (rc > 0) rc = cuda_fail(rc);
        if (rc) return rc;
        if (mode == JIT_MODE_DENSITY) {
            // a program writes its own record's row and the rows of the records that share it: no accumulators
            // to copy, and every row is written exactly once (write-only HBM traffic)
            std::map<uint32_t, std::vector<uint32_t>> followers;
            for (size_t i = 0; i + 1 < G.alias.size(); i += 2) followers[G.alias[i + 1]].push_back(G.alias[i]);
            for (uint32_t rec : cg.jit.h_slot_record) {
                cg.jit.h_row_begin.push_back((uint32_t)cg.jit.h_rows.size());
                cg.jit.h_rows.push_back(rec);
                auto it = followers.find(rec);
                if (it != followers.end()) cg.jit.h_rows.insert(cg.jit.h_rows.end(), it->second.begin(), it->second.end());
            }
            cg.jit.h_row_begin.push_back((uint32_t)cg.jit.h_rows.size());
            cg.alias.clear();
        }
        cp.groups.push_back(std::move(cg));
    }
    rc = instantiate_jit_plan(cp, out);
    if (rc) return rc;
    out->jit_compile_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    {
        std::lock_guard<std::mutex> lock(g_plan_cache_mutex);
        if (g_plan_cache.size() >= PLAN_CACHE_ENTRIES) {
            auto victim = g_plan_cache.begin();
            for (auto it = g_plan_cache.begin(); it != g_plan_cache.end(); ++it)
                if (it->second.stamp < victim->second.stamp) victim = it;
            g_plan_cache.erase(victim);
        }
        cp.stamp = ++g_plan_cache_clock;
        g_plan_cache.emplace(key, std::move(cp));
    }
    return KRIPKE_OK;
}

int build_jit_plan(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                   uint32_t cls, uint32_t flags, ScanPlan *out) {
    return build_jit_plan_mode(h, pairs, n_records, n, k, cls, flags, JIT_MODE_SCAN, out);
}

// Failure-density plan: every formula is a record of its own (one output row each), the graph is shared.
int build_density_plan(const kripke_programs *h, uint32_t n, uint32_t k, uint32_t cls, ScanPlan *out) {
    return build_jit_plan_mode(h, nullptr, h->n_formulas, n, k, cls, 0, JIT_MODE_DENSITY, out);
}

uint64_t plan_key(uint32_t n, uint32_t k, uint32_t cls, uint32_t flags, uint32_t engine, uint32_t shapes) {
    const uint32_t fl = flags & (KRIPKE_FULL_SWEEP | KRIPKE_NO_SHARING | KRIPKE_NO_SUBTERM_SHARING | KRIPKE_NO_GUARDED_ROOTS |
                                 KRIPKE_NO_BOX_DISTRIBUTION);
    return (uint64_t)n | ((uint64_t)k << 4) | ((uint64_t)cls << 8) | ((uint64_t)engine << 12) | ((uint64_t)fl << 16) |
           ((uint64_t)shapes << 32);
}

// Builds the plan of a record list with the engine the flags ask for.
int build_any_plan(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, uint32_t n, uint32_t k,
                   uint32_t cls, uint32_t flags, uint32_t engine, ScanPlan *out) {
    if (engine == ENGINE_JIT) {
        int rc = build_jit_plan(h, pairs, n_records, n, k, cls, flags, out);
        // AUTO falls back to the interpreted kernels when a record has no compiled layout
        if (rc != KRIPKE_EUNSUPPORTED || (flags & KRIPKE_KERNEL_MASK) == KRIPKE_KERNEL_JIT) return rc;
    }
    return build_scan_plan(h, pairs, n_records, n, k, reduced_shapes(n, k, cls, flags), out);
}

// The batch's plan for one shape (cached in the handle; synchronous on first use).
int single_plan(kripke_programs *h, uint32_t n, uint32_t k, uint32_t cls, uint32_t flags, const ScanPlan **out) {
    uint32_t engine = ENGINE_INTERPRETED;
    int rc = pick_engine(n, k, cls, flags, &engine);
    if (rc) return rc;
    // the interpreted plans depend on the class only through the usable shapes
    const uint64_t key = engine == ENGINE_JIT ? plan_key(n, k, cls, flags, engine, 0)
                                              : plan_key(n, k, 0, flags & (KRIPKE_FULL_SWEEP | KRIPKE_NO_SHARING), engine,
                                                         reduced_shapes(n, k, cls, flags));
    auto it = h->single.find(key);
    if (it == h->single.end()) {
        ScanPlan sp;
        rc = build_any_plan(h, nullptr, h->n_formulas, n, k, cls, flags, engine, &sp);
        if (rc) return rc;
        it = h->single.emplace(key, std::move(sp)).first;
    }
    *out = &it->second;
    return KRIPKE_OK;
}

// The plan of a pair list (cached in the handle: the size loop and repeated scans of one candidate set
// lower and compile once).  At most 8 lists are kept; the least recently used one is dropped.
int pair_plan(kripke_programs *h, const uint32_t *pairs, uint32_t n_pairs, uint32_t n, uint32_t k, uint32_t cls,
              uint32_t flags, kripke_programs::PairPlan **out) {
    uint32_t engine = ENGINE_INTERPRETED;
    int rc = pick_engine(n, k, cls, flags, &engine);
    if (rc) return rc;
    const uint64_t key = engine == ENGINE_JIT ? plan_key(n, k, cls, flags, engine, 0)
                                              : plan_key(n, k, 0, flags & (KRIPKE_FULL_SWEEP | KRIPKE_NO_SHARING), engine,
                                                         reduced_shapes(n, k, cls, flags));
    for (kripke_programs::PairPlan *pp : h->pair_plans)
        if (pp->key == key && pp->pairs.size() == 2 * (size_t)n_pairs &&
            std::equal(pp->pairs.begin(), pp->pairs.end(), pairs)) {
            pp->last_use = ++h->use_clock;
            *out = pp;
            return KRIPKE_OK;
        }
    if (h->pair_plans.size() >= 8) {
        size_t victim = 0;
        for (size_t i = 1; i < h->pair_plans.size(); ++i)
            if (h->pair_plans[i]->last_use < h->pair_plans[victim]->last_use) victim = i;
        if (h->has_last) CU(cudaEventSynchronize(h->done));          // it may still be in use on the device
        h->pair_plans[victim]->plan.release();
        cudaFree(h->pair_plans[victim]->d_pairs);
        delete h->pair_plans[victim];
        h->pair_plans.erase(h->pair_plans.begin() + victim);
    }
    kripke_programs::PairPlan *pp = new (std::nothrow) kripke_programs::PairPlan();
    if (!pp) return KRIPKE_ENOMEM;
    pp->pairs.assign(pairs, pairs + 2 * (size_t)n_pairs);
    pp->key = key;
    pp->last_use = ++h->use_clock;
    rc = build_any_plan(h, pairs, n_pairs, n, k, cls, flags, engine, &pp->plan);
    if (!rc) rc = upload(&pp->d_pairs, pp->pairs);
    if (rc) { pp->plan.release(); cudaFree(pp->d_pairs); delete pp; return rc; }
    h->pair_plans.push_back(pp);
    *out = pp;
    return KRIPKE_OK;
}

// ---- frame-list mode ----------------------------------------------------------------------------
// Lowers the records for scan_frames.cu: no derived leaves (the frames are data, nothing is
// thread-uniform), variables as written.
int build_list_plan(const kripke_programs *h, const uint32_t *pairs, uint32_t n_records, DevicePlan *out) {
    auto prog = [&](uint32_t f) { return &h->h_code[h->h_offsets[f]]; };
    auto plen = [&](uint32_t f) { return h->h_offsets[f + 1] - h->h_offsets[f]; };
    const uint8_t rename[KRIPKE_MAX_VARS] = {0, 1, 2, 3};
    // Records whose graphs coincide under the canonical variable order and polarity (jit.h) have the same counts
    // and the same first refuting list position on every list: one of them is scanned, the others copy its
    // accumulators before the finish step completes each record's own witness.
    std::vector<bool> skip(n_records, false);
    std::vector<uint32_t> alias;
    {
        Dag probe;
        std::map<std::pair<uint32_t, uint32_t>, uint32_t> seen;
        for (uint32_t r = 0; r < n_records; ++r) {
            const uint32_t fa = pairs ? pairs[2 * r] : r, fb = pairs ? pairs[2 * r + 1] : r;
            uint32_t sup;
            {
                Dag sd;
                sup = sd.support(sd.build(prog(fa), plen(fa), nullptr));
                if (pairs) sup |= sd.support(sd.build(prog(fb), plen(fb), nullptr));
            }
            uint8_t rn[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
            uint32_t neg = 0;
            canonical_rename(prog(fa), plen(fa), pairs ? prog(fb) : nullptr, pairs ? plen(fb) : 0u, sup, 1, 0, rn, &neg);
            uint32_t pa = probe.build(prog(fa), plen(fa), rn, neg);
            uint32_t pb = pairs ? probe.build(prog(fb), plen(fb), rn, neg) : UINT32_MAX;
            if (pairs && pb < pa) std::swap(pa, pb);
            auto it = seen.find(std::make_pair(pa, pb));
            if (it != seen.end()) { skip[r] = true; alias.push_back(r); alias.push_back(it->second); }
            else seen.emplace(std::make_pair(pa, pb), r);
        }
    }
    std::vector<Lowered> low(n_records);
    std::vector<bool> fits(n_records);
    for (uint32_t r = 0; r < n_records; ++r)
        if (!skip[r])
            fits[r] = pairs ? lower_pair(prog(pairs[2 * r]), plen(pairs[2 * r]), prog(pairs[2 * r + 1]),
                                         plen(pairs[2 * r + 1]), 0u, rename, &low[r])
                            : lower_single(prog(r), plen(r), 0u, rename, &low[r]);
    HostPlan hp;
    build_plan(low, fits, &hp, &skip);
    int rc = upload_plan(hp, out);
    if (!rc) rc = upload(&out->alias, alias);
    if (!rc) out->n_alias = (uint32_t)(alias.size() / 2);
    return rc;
}
int run_frames(kripke_programs *h, const DevicePlan &dp, const uint32_t *d_pairs, uint32_t n_records,
               uint32_t n, uint32_t k, const uint16_t *succ, uint64_t n_frames, uint64_t index_base,
               uint32_t flags, kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream) {
    if (n < 1 || n > KRIPKE_LIST_MAX_WORLDS || k != h->n_vars) return KRIPKE_EINVAL;
    if (k * n > KRIPKE_LIST_MAX_VAL_BITS) return KRIPKE_EUNSUPPORTED;
    if (flags & ~(KRIPKE_ACCUMULATE | KRIPKE_KERNEL_MASK)) return KRIPKE_EINVAL;
    const uint32_t family = flags & KRIPKE_KERNEL_MASK;
    if (n_frames && !succ) return KRIPKE_EINVAL;
    if (n_frames > (1ull << 40)) return KRIPKE_EUNSUPPORTED;
    if (n_records && (!counts_out || !witness_out)) return KRIPKE_EINVAL;
    if (family == KRIPKE_KERNEL_SLICED && dp.n_unfit) return KRIPKE_EUNSUPPORTED;
    h->last = kripke_run_info_t{};
    h->last.models_per_program = n_frames << (k * n);
    h->last.executed_models = (uint64_t)(n_records - (family == KRIPKE_KERNEL_SCALAR ? 0u : dp.n_alias)) * h->last.models_per_program;
    h->last.sliced_logic_ops_per_word = dp.n_modal * n * n + dp.n_bool * n + (uint64_t)dp.n_slots * (n + 1);
    h->last.logic_instr_per_frame = (double)h->last.sliced_logic_ops_per_word * (double)(1ull << (k * n)) / 32.0;
    h->last.popc_instr_per_frame = (double)dp.n_slots * (double)(1ull << (k * n)) / 32.0;
    h->last.kernel_family = family == KRIPKE_KERNEL_SCALAR ? 0 : 1;
    if (n_records == 0) return KRIPKE_OK;
    if (!h->done) CU(cudaEventCreateWithFlags(&h->done, cudaEventDisableTiming));
    if (h->has_last && h->last_stream != stream) CU(cudaStreamWaitEvent((cudaStream_t)stream, h->done, 0));
    if (n_records > h->accum_cap && h->has_last) CU(cudaEventSynchronize(h->done));
    int rc = ensure_accum(h, n_records);
    if (rc) return rc;
    FramesJob job;
    job.n = n; job.k = k; job.succ = succ; job.n_frames = n_frames; job.index_base = index_base;
    job.code = h->d_code; job.offsets = h->d_offsets; job.pairs = d_pairs;
    job.n_records = n_records; job.accum = h->d_accum;
    int e = launch_init(job.accum, n_records, stream);
    if (e) return cuda_fail(e);
    uint32_t launches = 1;
    if (family == KRIPKE_KERNEL_SCALAR) {
        if ((e = launch_frames_scalar(job, nullptr, n_records, stream, &launches))) return cuda_fail(e);
    } else {
        SlicedPlan sp;
        sp.ucode = dp.ucode; sp.slot_record = dp.slot_record; sp.n_slots = dp.n_slots;
        sp.stride = dp.stride; sp.max_need = 1; sp.model_shift = 0;
        for (uint32_t d = 1; d <= (uint32_t)UC_DMAX; ++d)
            if (dp.need_end[d] > dp.need_end[d - 1]) sp.max_need = d;
        if ((e = launch_frames(job, sp, stream, &launches))) return cuda_fail(e);
        if (dp.n_unfit && (e = launch_frames_scalar(job, dp.unfit, dp.n_unfit, stream, &launches))) return cuda_fail(e);
        if (dp.n_alias) {
            if ((e = launch_alias_accum(job.accum, dp.alias, dp.n_alias, stream))) return cuda_fail(e);
            ++launches;
        }
    }
    if ((e = launch_frames_finish(job, (flags & KRIPKE_ACCUMULATE) != 0, counts_out, witness_out, stream)))
        return cuda_fail(e);
    h->last.launches = launches + 1;
    CU(cudaEventRecord(h->done, (cudaStream_t)stream));
    h->last_stream = stream;
    h->has_last = true;
    return KRIPKE_OK;
}

}  // namespace

extern "C" {

int kripke_validity_bitmap(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                           uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                           uint32_t *bitmap_out, void *stream) {
    if (!programs) return KRIPKE_EINVAL;
    const kripke_programs *h = programs;
    if (n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || n_vars != h->n_vars || frame_class > KRIPKE_CLASS_S5)
        return KRIPKE_EINVAL;
    if (n_worlds * n_worlds + n_vars * n_worlds > KRIPKE_MAX_MODEL_BITS) return KRIPKE_EUNSUPPORTED;
    uint64_t csize = 0;
    int rc = class_size(n_worlds, frame_class, &csize);
    if (rc) return rc;
    if (frame_begin > csize || frame_count > csize - frame_begin) return KRIPKE_EINVAL;
    if (frame_count && h->n_formulas && !bitmap_out) return KRIPKE_EINVAL;
    ScanJob job;
    job.n = n_worlds; job.k = n_vars; job.cls = frame_class;
    job.frame_begin = frame_begin; job.frame_count = frame_count;
    if ((rc = class_table_device(n_worlds, frame_class, &job.class_table))) return rc;
    job.code = h->d_code; job.offsets = h->d_offsets; job.n_formulas = h->n_formulas;
    job.pairs = nullptr; job.n_records = h->n_formulas; job.accum = nullptr;
    const_cast<kripke_programs *>(programs)->aux_work = true;
    int e = launch_validity_bitmap(job, bitmap_out, stream);
    return e ? cuda_fail(e) : KRIPKE_OK;
}

int kripke_condition_bitmap(uint32_t n_worlds, uint32_t condition, uint32_t frame_class, uint64_t frame_begin,
                            uint64_t frame_count, uint32_t *bitmap_out, void *stream) {
    if (n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || condition >= KRIPKE_COND_COUNT || frame_class > KRIPKE_CLASS_S5)
        return KRIPKE_EINVAL;
    uint64_t csize = 0;
    int rc = class_size(n_worlds, frame_class, &csize);
    if (rc) return rc;
    if (frame_begin > csize || frame_count > csize - frame_begin) return KRIPKE_EINVAL;
    if (frame_count && !bitmap_out) return KRIPKE_EINVAL;
    const uint64_t *table = nullptr;
    if ((rc = class_table_device(n_worlds, frame_class, &table))) return rc;
    int e = launch_condition_bitmap(n_worlds, condition, frame_class, table, frame_begin, frame_count, bitmap_out, stream);
    return e ? cuda_fail(e) : KRIPKE_OK;
}

int kripke_failure_density(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                           uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                           uint32_t *counts_out, void *stream) {
    if (!programs) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    if (n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || n_vars != h->n_vars || frame_class > KRIPKE_CLASS_S5)
        return KRIPKE_EINVAL;
    if (n_vars * n_worlds > KRIPKE_LIST_MAX_VAL_BITS) return KRIPKE_EUNSUPPORTED;
    uint64_t csize = 0;
    int rc = class_size(n_worlds, frame_class, &csize);
    if (rc) return rc;
    if (frame_begin > csize || frame_count > csize - frame_begin) return KRIPKE_EINVAL;
    if (frame_count && h->n_formulas && !counts_out) return KRIPKE_EINVAL;
    h->aux_work = true;
    ScanJob job;
    job.n = n_worlds; job.k = n_vars; job.cls = frame_class;
    job.frame_begin = frame_begin; job.frame_count = frame_count;
    if ((rc = class_table_device(n_worlds, frame_class, &job.class_table))) return rc;
    job.code = h->d_code; job.offsets = h->d_offsets; job.n_formulas = h->n_formulas;
    job.pairs = nullptr; job.n_records = h->n_formulas; job.accum = nullptr;
    h->last = kripke_run_info_t{};
    h->last.models_per_program = frame_count << (n_vars * n_worlds);
    if (frame_count == 0 || h->n_formulas == 0) return KRIPKE_OK;
    // Compiled bit-sliced kernels when every variable-count group has a density layout and the rows can be
    // written with 16-byte stores; the scalar kernel (thread = frame, one model per iteration) otherwise and on
    // the ragged ends of the range.
    bool compiled = jit_density_layout(n_worlds, n_vars, frame_class, nullptr) && frame_count % 4 == 0 &&
                    frame_begin % 4 == 0 && (reinterpret_cast<uintptr_t>(counts_out) & 15u) == 0;
    const ScanPlan *plan = nullptr;
    if (compiled) {
        const uint64_t key = plan_key(n_worlds, n_vars, frame_class, 0, ENGINE_JIT, 0);
        auto it = h->density.find(key);
        if (it == h->density.end()) {
            ScanPlan sp;
            rc = build_density_plan(h, n_worlds, n_vars, frame_class, &sp);
            if (rc == KRIPKE_EUNSUPPORTED) compiled = false;
            else if (rc) return rc;
            else it = h->density.emplace(key, std::move(sp)).first;
        }
        if (compiled) plan = &it->second;
    }
    int e = 0;
    uint32_t launches = 0;
    if (!compiled) {
        if ((e = launch_failure_density(job, nullptr, counts_out, frame_count, 0, stream))) return cuda_fail(e);
        h->last.launches = 1;
        return KRIPKE_OK;
    }
    h->last.kernel_family = 2;
    h->last.jit_compile_seconds = plan->jit_compile_seconds;
    for (const GroupPlan &g : plan->groups) {
        const uint64_t fpu = 1ull << g.jit.lay.unit_frames_log2;
        uint64_t ab = (frame_begin + fpu - 1) / fpu * fpu, ae = (frame_begin + frame_count) / fpu * fpu;
        if (ae <= ab) ab = ae = frame_begin;
        const double words = (double)(1ull << (g.k_eff * n_worlds)) / 32.0;
        h->last.logic_instr_per_frame += g.jit.stats.logic_ops_per_word * words;
        h->last.jit_programs += g.jit.n_slots;
        if (ae > ab) {
            ScanJob rj = job;
            rj.k = g.k_eff; rj.frame_begin = ab; rj.frame_count = ae - ab;
            JitDensityOut out{counts_out, frame_count, frame_begin};
            if ((e = jit_launch_group(rj, g.jit, (n_vars - g.k_eff) * n_worlds, &out, stream, &launches))) return cuda_fail(e);
        }
        // ragged ends: the scalar kernel on this group's records only
        for (int side = 0; side < 2; ++side) {
            ScanJob sj = job;
            sj.frame_begin = side ? ae : frame_begin;
            sj.frame_count = side ? frame_begin + frame_count - ae : ab - frame_begin;
            if (sj.frame_count == 0) continue;
            if ((e = launch_failure_density_records(sj, g.jit.d_slot_record, g.jit.n_slots, g.jit.d_row_begin, g.jit.d_rows,
                                                    counts_out, frame_count, sj.frame_begin - frame_begin, stream)))
                return cuda_fail(e);
            ++launches;
        }
    }
    h->last.launches = launches;
    return KRIPKE_OK;
}

int kripke_failure_density_frames(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                                  const uint16_t *succ, uint64_t n_frames, uint32_t *counts_out, void *stream) {
    if (!programs) return KRIPKE_EINVAL;
    const kripke_programs *h = programs;
    if (n_worlds < 1 || n_worlds > KRIPKE_LIST_MAX_WORLDS || n_vars != h->n_vars) return KRIPKE_EINVAL;
    if (n_vars * n_worlds > KRIPKE_LIST_MAX_VAL_BITS) return KRIPKE_EUNSUPPORTED;
    if (n_frames && (!succ || (h->n_formulas && !counts_out))) return KRIPKE_EINVAL;
    ScanJob job;
    job.n = n_worlds; job.k = n_vars; job.cls = KRIPKE_CLASS_K;
    job.frame_begin = 0; job.frame_count = n_frames; job.class_table = nullptr;
    job.code = h->d_code; job.offsets = h->d_offsets; job.n_formulas = h->n_formulas;
    job.pairs = nullptr; job.n_records = h->n_formulas; job.accum = nullptr;
    const_cast<kripke_programs *>(programs)->aux_work = true;
    int e = launch_failure_density(job, succ, counts_out, n_frames, 0, stream);
    return e ? cuda_fail(e) : KRIPKE_OK;
}

int kripke_frames_generate(uint32_t generator, uint32_t n_worlds, uint64_t n_frames, uint64_t seed, uint16_t *succ_out,
                           void *stream) {
    if (generator >= KRIPKE_GEN_COUNT || n_worlds < 1 || n_worlds > KRIPKE_LIST_MAX_WORLDS) return KRIPKE_EINVAL;
    if (n_frames > (1ull << 32)) return KRIPKE_EUNSUPPORTED;
    if (n_frames && !succ_out) return KRIPKE_EINVAL;
    int e = launch_frames_generate(generator, n_worlds, n_frames, seed, succ_out, stream);
    return e ? cuda_fail(e) : KRIPKE_OK;
}

int kripke_signatures(const kripke_programs_t *programs, uint32_t n_vars, uint32_t n_max, uint64_t *sig_out,
                      void *stream) {
    if (!programs) return KRIPKE_EINVAL;
    const kripke_programs *h = programs;
    if (n_vars != h->n_vars || n_max < 1 || n_max > 4) return KRIPKE_EINVAL;
    if (n_max * n_max + n_vars * n_max > 40) return KRIPKE_EUNSUPPORTED;
    if (h->n_formulas && !sig_out) return KRIPKE_EINVAL;
    const_cast<kripke_programs *>(programs)->aux_work = true;
    int e = launch_signatures(n_vars, n_max, h->d_code, h->d_offsets, h->n_formulas, sig_out, stream);
    return e ? cuda_fail(e) : KRIPKE_OK;
}

int kripke_frames_from_bitmap(uint32_t n_worlds, uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                              const uint32_t *bitmap, uint16_t *succ_out, uint64_t capacity, uint64_t *count_out,
                              void *stream) {
    if (n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || frame_class > KRIPKE_CLASS_S5 || !count_out) return KRIPKE_EINVAL;
    uint64_t csize = 0;
    int rc = class_size(n_worlds, frame_class, &csize);
    if (rc) return rc;
    if (frame_begin > csize || frame_count > csize - frame_begin) return KRIPKE_EINVAL;
    if (frame_count && (!bitmap || (capacity && !succ_out))) return KRIPKE_EINVAL;
    const uint64_t *table = nullptr;
    if ((rc = class_table_device(n_worlds, frame_class, &table))) return rc;
    int e = launch_frames_from_bitmap(n_worlds, frame_class, table, frame_begin, frame_count, bitmap, succ_out,
                                      capacity, count_out, stream);
    return e ? cuda_fail(e) : KRIPKE_OK;
}

int kripke_match_bitmaps(const uint32_t *bitmaps, uint32_t n_records, uint64_t words, const uint32_t *library,
                         uint32_t n_library, uint32_t *match_out, void *stream) {
    if (n_records && (!match_out || (words && !bitmaps))) return KRIPKE_EINVAL;
    if (n_library && words && !library) return KRIPKE_EINVAL;
    int e = launch_match_bitmaps(bitmaps, n_records, words, library, n_library, match_out, stream);
    return e ? cuda_fail(e) : KRIPKE_OK;
}

int kripke_eval_frames(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                       const uint16_t *succ, uint64_t n_frames, uint64_t index_base, uint32_t flags,
                       kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream) {
    if (!programs) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    if (!h->list_single_built) {
        int rc = build_list_plan(h, nullptr, h->n_formulas, &h->list_single);
        if (rc) return rc;
        h->list_single_built = true;
    }
    return run_frames(h, h->list_single, nullptr, h->n_formulas, n_worlds, n_vars, succ, n_frames, index_base,
                      flags, counts_out, witness_out, stream);
}

int kripke_distinguish_pairs_frames(const kripke_programs_t *programs, const uint32_t *pairs,
                                    uint32_t n_pairs, uint32_t n_worlds, uint32_t n_vars,
                                    const uint16_t *succ, uint64_t n_frames, uint64_t index_base,
                                    uint32_t flags, kripke_count_t *counts_out,
                                    kripke_witness_t *witness_out, void *stream) {
    if (!programs || (n_pairs && !pairs)) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    for (uint32_t i = 0; i < 2 * n_pairs; ++i)
        if (pairs[i] >= h->n_formulas) return KRIPKE_EINVAL;
    const bool same = h->list_pair_built && h->list_pair_key.size() == 2 * (size_t)n_pairs &&
                      std::equal(h->list_pair_key.begin(), h->list_pair_key.end(), pairs);
    if (!same) {
        if (h->has_last) CU(cudaEventSynchronize(h->done));   // the previous call's plan may still be in use
        h->list_pair_built = false;
        int rc = build_list_plan(h, pairs, n_pairs, &h->list_pair);
        if (rc) return rc;
        if (n_pairs > h->pairs_cap) {
            cudaFree(h->d_pairs);
            h->d_pairs = nullptr; h->pairs_cap = 0;
            CU(cudaMalloc((void **)&h->d_pairs, (size_t)2 * n_pairs * sizeof(uint32_t)));
            h->pairs_cap = n_pairs;
        }
        if (n_pairs) CU(cudaMemcpy(h->d_pairs, pairs, (size_t)2 * n_pairs * sizeof(uint32_t), cudaMemcpyHostToDevice));
        h->list_pair_key.assign(pairs, pairs + 2 * (size_t)n_pairs);
        h->list_pair_built = true;
    }
    return run_frames(h, h->list_pair, h->d_pairs, n_pairs, n_worlds, n_vars, succ, n_frames, index_base, flags,
                      counts_out, witness_out, stream);
}

const char *kripke_version(void) { return "kripke-b200 0.2 (sm_100a)"; }

int kripke_last_cuda_error(void) { return g_last_cuda_error; }

int kripke_validate_programs(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                             uint32_t n_vars, uint32_t *max_stack_out) {
    return validate_programs(code, offsets, n_formulas, n_vars, max_stack_out);
}

int kripke_class_size(uint32_t n_worlds, uint32_t frame_class, uint64_t *size_out) {
    if (!size_out) return KRIPKE_EINVAL;
    return class_size(n_worlds, frame_class, size_out);
}

int kripke_programs_create(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                           uint32_t n_vars, kripke_programs_t **programs_out) {
    if (!programs_out) return KRIPKE_EINVAL;
    *programs_out = nullptr;
    int rc = validate_programs(code, offsets, n_formulas, n_vars, nullptr);
    if (rc) return rc;
    kripke_programs *h = new (std::nothrow) kripke_programs();
    if (!h) return KRIPKE_ENOMEM;
    ++g_live_handles;
    h->n_formulas = n_formulas;
    h->n_vars = n_vars;
    h->h_offsets.assign(offsets, offsets + n_formulas + 1);
    h->h_code.assign(code + offsets[0], code + offsets[n_formulas]);
    const uint32_t base = offsets[0];
    for (auto &o : h->h_offsets) o -= base;
    h->f_modal.assign(n_formulas, 0); h->f_binary.assign(n_formulas, 0); h->f_vars.assign(n_formulas, 0);
    for (uint32_t f = 0; f < n_formulas; ++f)
        for (uint32_t i = h->h_offsets[f]; i < h->h_offsets[f + 1]; ++i) {
            const uint8_t c = h->h_code[i];
            if (c == KRIPKE_OP_BOX || c == KRIPKE_OP_DIA) ++h->f_modal[f];
            else if (c >= KRIPKE_OP_AND) ++h->f_binary[f];
            else if (c >= KRIPKE_OP_VAR0 && c < KRIPKE_OP_NOT) h->f_vars[f] |= 1u << (c - KRIPKE_OP_VAR0);
        }
    if (h->h_code.empty()) h->h_code.push_back(0);
    if ((rc = upload(&h->d_code, h->h_code)) || (rc = upload(&h->d_offsets, h->h_offsets))) {
        kripke_programs_destroy(h);
        return rc;
    }
    *programs_out = h;
    return KRIPKE_OK;
}

int kripke_programs_destroy(kripke_programs_t *h) {
    if (!h) return KRIPKE_OK;
    // A handle that only ran scans waits for its own last scan (every scan records h->done, on every exit path)
    // and leaves other handles' streams alone; one that also enqueued other work on its memory, possibly on
    // several streams, has no single event for it and waits for the device.
    if (h->aux_work) cudaDeviceSynchronize();
    else if (h->has_last && h->done) cudaEventSynchronize(h->done);
    for (auto &kv : h->single) kv.second.release();
    for (auto &kv : h->density) kv.second.release();
    for (kripke_programs::PairPlan *pp : h->pair_plans) { pp->plan.release(); cudaFree(pp->d_pairs); delete pp; }
    if (h->done) cudaEventDestroy(h->done);
    h->list_single.release(); h->list_pair.release();
    cudaFree(h->d_code); cudaFree(h->d_offsets); cudaFree(h->d_pairs); cudaFree(h->d_accum);
    cudaFree(h->d_tmp_counts); cudaFree(h->d_tmp_wit);
    delete h;
    --g_live_handles;
    return KRIPKE_OK;
}

int kripke_jit_cache_clear(uint32_t *modules_unloaded_out) {
    if (modules_unloaded_out) *modules_unloaded_out = 0;
    if (g_live_handles.load() > 0) return KRIPKE_EINVAL;      // their cached plans point into the modules
    CU(cudaDeviceSynchronize());                              // a destroyed handle's last scan may still be running
    {
        std::lock_guard<std::mutex> lock(g_plan_cache_mutex);
        g_plan_cache.clear();
    }
    const size_t n = jit_cache_clear();
    if (modules_unloaded_out) *modules_unloaded_out = (uint32_t)n;
    return KRIPKE_OK;
}

int kripke_eval_batch_range(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                            uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                            uint32_t flags, kripke_count_t *counts_out, kripke_witness_t *witness_out,
                            void *stream) {
    if (!programs) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    // every argument is checked before a plan is built or cached
    int rc = check_scan_args(h, h->n_formulas, n_worlds, n_vars, frame_class, frame_begin, frame_count, flags,
                             counts_out, witness_out);
    if (rc) return rc;
    const ScanPlan *plan = nullptr;
    if ((rc = single_plan(h, n_worlds, n_vars, frame_class, flags, &plan))) return rc;
    return run_scan(h, *plan, nullptr, nullptr, h->n_formulas, n_worlds, n_vars, frame_class, frame_begin,
                    frame_count, flags, counts_out, witness_out, stream);
}

int kripke_eval_batch(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                      uint32_t frame_class, kripke_count_t *counts_out, kripke_witness_t *witness_out,
                      void *stream) {
    uint64_t csize = 0;
    int rc = class_size(n_worlds, frame_class, &csize);
    if (rc) return rc;
    return kripke_eval_batch_range(programs, n_worlds, n_vars, frame_class, 0, csize, 0, counts_out,
                                   witness_out, stream);
}

int kripke_distinguish_pairs(const kripke_programs_t *programs, const uint32_t *pairs, uint32_t n_pairs,
                             uint32_t n_worlds, uint32_t n_vars, uint32_t frame_class,
                             uint64_t frame_begin, uint64_t frame_count, uint32_t flags,
                             kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream) {
    if (!programs || (n_pairs && !pairs)) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    for (uint32_t i = 0; i < 2 * n_pairs; ++i)
        if (pairs[i] >= h->n_formulas) return KRIPKE_EINVAL;
    int rc = check_scan_args(h, n_pairs, n_worlds, n_vars, frame_class, frame_begin, frame_count, flags, counts_out,
                             witness_out);
    if (rc) return rc;
    kripke_programs::PairPlan *pp = nullptr;
    if ((rc = pair_plan(h, pairs, n_pairs, n_worlds, n_vars, frame_class, flags, &pp))) return rc;
    return run_scan(h, pp->plan, pp->pairs.data(), pp->d_pairs, n_pairs, n_worlds, n_vars, frame_class, frame_begin,
                    frame_count, flags, counts_out, witness_out, stream);
}

int kripke_minimal_refutation(const kripke_programs_t *programs, uint32_t n_vars, uint32_t frame_class,
                              uint32_t n_max, uint32_t *size_out, kripke_count_t *counts_out,
                              kripke_witness_t *witness_out, void *stream) {
    if (!programs || n_max < 1 || n_max > KRIPKE_MAX_WORLDS) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    const uint32_t B = h->n_formulas;
    if (B && (!size_out || !counts_out || !witness_out)) return KRIPKE_EINVAL;
    h->aux_work = true;                       // the record kernel reads d_tmp_* after the scan's event
    if (B > h->tmp_cap) {
        cudaFree(h->d_tmp_counts); cudaFree(h->d_tmp_wit);
        h->d_tmp_counts = nullptr; h->d_tmp_wit = nullptr; h->tmp_cap = 0;
        CU(cudaMalloc((void **)&h->d_tmp_counts, (size_t)B * sizeof(kripke_count_t)));
        CU(cudaMalloc((void **)&h->d_tmp_wit, (size_t)B * sizeof(kripke_witness_t)));
        h->tmp_cap = B;
    }
    for (uint32_t n = 1; n <= n_max; ++n) {
        int rc = kripke_eval_batch(h, n, n_vars, frame_class, h->d_tmp_counts, h->d_tmp_wit, stream);
        if (rc) return rc;
        int e = launch_record_size(n, B, h->d_tmp_counts, h->d_tmp_wit, size_out, counts_out, witness_out, stream);
        if (e) return cuda_fail(e);
    }
    return KRIPKE_OK;
}

int kripke_pairs_separation(const kripke_programs_t *programs, const uint32_t *pairs, uint32_t n_pairs,
                            uint32_t n_vars, uint32_t n_max, uint64_t chunk_frames,
                            uint32_t *size_out, kripke_witness_t *witness_out, void *stream) {
    if (!programs || n_max < 1 || n_max > KRIPKE_MAX_WORLDS || chunk_frames == 0) return KRIPKE_EINVAL;
    if (n_pairs && (!pairs || !size_out || !witness_out)) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    std::vector<uint32_t> active(n_pairs);          // indices of the pairs not separated yet
    for (uint32_t j = 0; j < n_pairs; ++j) {
        active[j] = j;
        size_out[j] = 0;
        witness_out[j].frame = KRIPKE_NO_WITNESS; witness_out[j].valuation = 0; witness_out[j].world = 0;
    }
    kripke_count_t *d_counts = nullptr;
    kripke_witness_t *d_wit = nullptr;
    if (n_pairs) {
        CU(cudaMalloc((void **)&d_counts, (size_t)n_pairs * sizeof(kripke_count_t)));
        cudaError_t e = cudaMalloc((void **)&d_wit, (size_t)n_pairs * sizeof(kripke_witness_t));
        if (e != cudaSuccess) { cudaFree(d_counts); return cuda_fail((int)e); }
    }
    std::vector<kripke_count_t> hc(n_pairs);
    std::vector<kripke_witness_t> hw(n_pairs);
    std::vector<uint32_t> sub, listed;               // the pair list of the current plan and the pairs it holds
    int rc = KRIPKE_OK;
    for (uint32_t n = 1; n <= n_max && rc == KRIPKE_OK && !active.empty(); ++n) {
        const uint64_t total = 1ull << (n * n);
        listed.clear();
        for (uint64_t begin = 0; begin < total && rc == KRIPKE_OK && !active.empty(); begin += chunk_frames) {
            const uint64_t count = std::min<uint64_t>(chunk_frames, total - begin);
            // the records are lowered (and compiled) once per size; a new list is made only when at least half
            // of the listed pairs have left the scan, so a long chunked size costs O(log P) plans
            if (listed.empty() || 2 * active.size() <= listed.size()) {
                listed = active;
                sub.resize(2 * listed.size());
                for (size_t a = 0; a < listed.size(); ++a) {
                    sub[2 * a] = pairs[2 * listed[a]];
                    sub[2 * a + 1] = pairs[2 * listed[a] + 1];
                }
            }
            rc = kripke_distinguish_pairs(h, sub.data(), (uint32_t)listed.size(), n, n_vars, KRIPKE_CLASS_K, begin,
                                          count, 0, d_counts, d_wit, stream);
            if (rc) break;
            cudaError_t e = cudaMemcpyAsync(hc.data(), d_counts, listed.size() * sizeof(kripke_count_t),
                                            cudaMemcpyDeviceToHost, (cudaStream_t)stream);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(hw.data(), d_wit, listed.size() * sizeof(kripke_witness_t),
                                    cudaMemcpyDeviceToHost, (cudaStream_t)stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
            if (e != cudaSuccess) { rc = cuda_fail((int)e); break; }
            std::vector<uint32_t> still;
            for (size_t a = 0; a < listed.size(); ++a) {
                const uint32_t j = listed[a];
                if (size_out[j] != 0) continue;                       // separated in an earlier chunk
                if (hc[a].refuting_models != 0) {
                    size_out[j] = n;
                    witness_out[j] = hw[a];
                } else {
                    still.push_back(j);
                }
            }
            active.swap(still);
        }
    }
    cudaFree(d_counts);
    cudaFree(d_wit);
    return rc;
}

int kripke_eval_batch_host(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                           uint32_t n_worlds, uint32_t n_vars, uint32_t frame_class,
                           kripke_count_t *counts_host, kripke_witness_t *witness_host) {
    if (n_formulas && (!counts_host || !witness_host)) return KRIPKE_EINVAL;
    kripke_programs_t *h = nullptr;
    int rc = kripke_programs_create(code, offsets, n_formulas, n_vars, &h);
    if (rc) return rc;
    kripke_count_t *d_counts = nullptr;
    kripke_witness_t *d_wit = nullptr;
    cudaError_t e = cudaSuccess;
    if (n_formulas) {
        e = cudaMalloc((void **)&d_counts, n_formulas * sizeof(kripke_count_t));
        if (e == cudaSuccess) e = cudaMalloc((void **)&d_wit, n_formulas * sizeof(kripke_witness_t));
    }
    if (e == cudaSuccess) {
        rc = kripke_eval_batch(h, n_worlds, n_vars, frame_class, d_counts, d_wit, nullptr);
        if (rc == KRIPKE_OK && n_formulas) {
            e = cudaMemcpy(counts_host, d_counts, n_formulas * sizeof(kripke_count_t), cudaMemcpyDeviceToHost);
            if (e == cudaSuccess)
                e = cudaMemcpy(witness_host, d_wit, n_formulas * sizeof(kripke_witness_t), cudaMemcpyDeviceToHost);
        }
    }
    cudaFree(d_counts);
    cudaFree(d_wit);
    kripke_programs_destroy(h);
    if (e != cudaSuccess) return cuda_fail((int)e);
    return rc;
}

int kripke_last_run_info(const kripke_programs_t *programs, kripke_run_info_t *info_out) {
    if (!programs || !info_out) return KRIPKE_EINVAL;
    *info_out = programs->last;
    return KRIPKE_OK;
}

static int witness_keys(bool to_keys, const void *src, uint32_t n_records, uint32_t n, uint32_t k, void *dst,
                        void *stream) {
    if (n < 1 || n > KRIPKE_MAX_WORLDS || k > KRIPKE_MAX_VARS || n * n + k * n > KRIPKE_MAX_MODEL_BITS) return KRIPKE_EINVAL;
    if (n_records && (!src || !dst)) return KRIPKE_EINVAL;
    int e = launch_witness_keys(to_keys, src, n_records, k * n, dst, stream);
    if (e) return cuda_fail(e);
    return KRIPKE_OK;
}

int kripke_witness_to_keys(const kripke_witness_t *witness, uint32_t n_records, uint32_t n_worlds,
                           uint32_t n_vars, uint64_t *keys_out, void *stream) {
    return witness_keys(true, witness, n_records, n_worlds, n_vars, keys_out, stream);
}

int kripke_keys_to_witness(const uint64_t *keys, uint32_t n_records, uint32_t n_worlds, uint32_t n_vars,
                           kripke_witness_t *witness_out, void *stream) {
    return witness_keys(false, keys, n_records, n_worlds, n_vars, witness_out, stream);
}

int kripke_debug_lower(const uint8_t *code_a, uint32_t len_a, const uint8_t *code_b, uint32_t len_b,
                       uint32_t n_vars, uint32_t leaf_mode, uint16_t *ucode_out, uint32_t cap,
                       uint32_t *need_out) {
    if (!code_a || !ucode_out) return KRIPKE_EINVAL;
    const uint32_t offs_a[2] = {0, len_a}, offs_b[2] = {0, len_b};
    int rc = validate_programs(code_a, offs_a, 1, n_vars, nullptr);
    if (rc == KRIPKE_OK && code_b) rc = validate_programs(code_b, offs_b, 1, n_vars, nullptr);
    if (rc) return rc;
    Lowered low;
    if (leaf_mode > (LOWER_LEAF_DEAD | LOWER_LEAF_P | LOWER_FUSE)) return KRIPKE_EINVAL;
    const bool fits = code_b ? lower_pair(code_a, len_a, code_b, len_b, leaf_mode, nullptr, &low)
                             : lower_single(code_a, len_a, leaf_mode, nullptr, &low);
    if (need_out) *need_out = (uint32_t)low.need;
    if (!fits) return KRIPKE_EUNSUPPORTED;
    if (low.ucode.size() > cap) return KRIPKE_EINVAL;
    std::memcpy(ucode_out, low.ucode.data(), low.ucode.size() * sizeof(uint16_t));
    return (int)low.ucode.size();
}

int kripke_jit_configure(uint32_t max_programs_per_kernel, uint32_t min_blocks_per_sm) {
    if (max_programs_per_kernel < 1 || max_programs_per_kernel > 160) return KRIPKE_EINVAL;
    if (min_blocks_per_sm < 1 || min_blocks_per_sm > 8) return KRIPKE_EINVAL;
    g_jit_max_programs = max_programs_per_kernel;
    g_jit_min_blocks = min_blocks_per_sm;
    return KRIPKE_OK;
}

int kripke_debug_jit_source(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas, uint32_t n_vars,
                            const uint32_t *pairs, uint32_t n_pairs,
                            uint32_t n_worlds, uint32_t frame_class, uint32_t flags, uint32_t group_vars,
                            uint32_t kernel_index, int compile, char *source_out, uint64_t cap,
                            uint32_t *n_kernels_out, uint64_t *logic_ops_per_word_out, uint64_t *cubin_bytes_out) {
    if (n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || frame_class > KRIPKE_CLASS_S5) return KRIPKE_EINVAL;
    int rc0 = validate_programs(code, offsets, n_formulas, n_vars, nullptr);
    if (rc0) return rc0;
    kripke_programs tmp;                       // host fields only: nothing here touches a device
    tmp.n_formulas = n_formulas; tmp.n_vars = n_vars;
    tmp.h_offsets.assign(offsets, offsets + n_formulas + 1);
    tmp.h_code.assign(code + offsets[0], code + offsets[n_formulas]);
    for (auto &o : tmp.h_offsets) o -= offsets[0];
    const kripke_programs *h = &tmp;
    if (group_vars > h->n_vars) return KRIPKE_EINVAL;
    for (uint32_t i = 0; pairs && i < 2 * n_pairs; ++i)
        if (pairs[i] >= h->n_formulas) return KRIPKE_EINVAL;
    std::vector<JitGroupHost> groups;
    const uint32_t mode = (compile & 2) ? JIT_MODE_DENSITY : JIT_MODE_SCAN;
    if (mode == JIT_MODE_DENSITY && pairs) return KRIPKE_EINVAL;
    int rc = jit_group_records(h, pairs, pairs ? n_pairs : h->n_formulas, n_worlds, h->n_vars, frame_class, flags,
                               mode, &groups);
    if (rc) return rc;
    const JitGroupHost &G = groups[group_vars];
    JitLayout lay;
    if (!(mode == JIT_MODE_DENSITY ? jit_density_layout(n_worlds, group_vars, frame_class, &lay)
                                   : jit_layout(n_worlds, group_vars, frame_class, &lay)))
        return KRIPKE_EUNSUPPORTED;
    std::vector<std::vector<uint32_t>> parts;
    if (mode == JIT_MODE_DENSITY) {
        for (uint32_t r = 0; r < G.roots.size(); ++r) {
            if (r % 32 == 0) parts.emplace_back();
            parts.back().push_back(r);
        }
    } else {
        parts = jit_partition(G.dag, G.roots, lay, g_jit_max_programs);
    }
    if (n_kernels_out) *n_kernels_out = (uint32_t)parts.size();
    if (logic_ops_per_word_out) *logic_ops_per_word_out = 0;
    if (cubin_bytes_out) *cubin_bytes_out = 0;
    if (kernel_index >= parts.size()) return parts.empty() ? KRIPKE_OK : KRIPKE_EINVAL;
    std::vector<JitRoot> rs;
    for (uint32_t r : parts[kernel_index]) rs.push_back(G.roots[r]);
    JitEmitStats st;
    const std::string src = jit_emit_kernel(G.dag, lay, rs, 128, g_jit_min_blocks, mode, &st);
    if (logic_ops_per_word_out) *logic_ops_per_word_out = (uint64_t)(st.logic_ops_per_word + 0.5);
    if (compile & 1) {
        std::string log;
        size_t bytes = 0;
        if ((rc = jit_compile_only(src, &log, &bytes))) return rc;
        if (cubin_bytes_out) *cubin_bytes_out = bytes;
    }
    if (source_out && cap) {
        const size_t m = std::min<size_t>(src.size(), (size_t)cap - 1);
        std::memcpy(source_out, src.data(), m);
        source_out[m] = 0;
    }
    return (int)std::min<size_t>(src.size(), 0x7FFFFFFF);
}

int kripke_debug_batch_refuted(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas, uint32_t n_vars,
                               uint32_t n_worlds, uint32_t frame_class, uint32_t flags, const uint32_t *succ,
                               const uint32_t *val, uint8_t *refuted_out) {
    if (!succ || !refuted_out || n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || frame_class > KRIPKE_CLASS_S5 ||
        (n_vars && !val))
        return KRIPKE_EINVAL;
    int rc = validate_programs(code, offsets, n_formulas, n_vars, nullptr);
    if (rc) return rc;
    kripke_programs tmp;                       // host fields only
    tmp.n_formulas = n_formulas; tmp.n_vars = n_vars;
    tmp.h_offsets.assign(offsets, offsets + n_formulas + 1);
    tmp.h_code.assign(code + offsets[0], code + offsets[n_formulas]);
    for (auto &o : tmp.h_offsets) o -= offsets[0];
    std::vector<JitGroupHost> groups;
    std::vector<JitRecordInfo> info;
    rc = jit_group_records(&tmp, nullptr, n_formulas, n_worlds, n_vars, frame_class, flags, JIT_MODE_SCAN, &groups, &info);
    if (rc) return rc;
    int rewrites = 0;
    for (const JitGroupHost &G : groups) rewrites += (int)G.opt.rewrites;
    for (uint32_t r = 0; r < n_formulas; ++r) {
        const JitRecordInfo &ri = info[r];
        uint32_t pv[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
        for (uint32_t v = 0; v < n_vars; ++v)
            if ((ri.support >> v) & 1u) pv[ri.rename[v]] = ((ri.neg >> v) & 1u) ? ~val[v] : val[v];
        const JitGroupHost &G = groups[ri.group];
        refuted_out[r] = jit_root_refuted(G.dag, G.roots[ri.slot], n_worlds, succ, pv) ? 1 : 0;
    }
    return rewrites;
}

int kripke_debug_dag_truth(const uint8_t *code, uint32_t len, uint32_t n_vars, uint32_t n_worlds,
                           const uint32_t *succ, const uint32_t *val, uint32_t *truth_out) {
    if (!code || !succ || !truth_out || n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || (n_vars && !val)) return KRIPKE_EINVAL;
    const uint32_t offs[2] = {0, len};
    int rc = validate_programs(code, offs, 1, n_vars, nullptr);
    if (rc) return rc;
    // evaluated under the canonical variable order, with the valuation permuted the same way
    uint8_t rename[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
    uint32_t sup;
    {
        Dag sd;
        sup = sd.support(sd.build(code, len, nullptr));
    }
    canonical_rename(code, len, nullptr, 0, sup, n_worlds, 0, rename);
    uint32_t pv[KRIPKE_MAX_VARS] = {0, 0, 0, 0};
    for (uint32_t v = 0; v < n_vars; ++v)
        if ((sup >> v) & 1u) pv[rename[v]] = val[v];
    Dag d;
    const uint32_t root = d.build(code, len, rename);
    *truth_out = d.eval(root, n_worlds, succ, pv);
    return (int)d.nodes.size();
}

int kripke_calibrate_int32(uint32_t variant, double *thread_instr_per_s_out, double *elapsed_ms_out,
                           void *stream) {
    if (variant > 5 || !thread_instr_per_s_out) return KRIPKE_EINVAL;
    int e = run_calibration(variant, thread_instr_per_s_out, elapsed_ms_out, stream);
    if (e) return cuda_fail(e);
    return KRIPKE_OK;
}

}  // extern "C"
