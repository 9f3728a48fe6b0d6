// api.cpp - the C ABI of include/kripke.h: argument checking, program staging (H1), class tables
// (H2), kernel selection and launch sequencing.  All compute runs in the CUDA kernels of this
// library; there is no CPU evaluation path here.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <tuple>

#include "internal.h"

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

// A lowered set of records for the sliced kernel plus the list of records it cannot run.
struct HostPlan {
    std::vector<uint16_t> ucode;
    std::vector<uint32_t> slot_record;
    std::vector<uint32_t> unfit;
    uint32_t stride = 2;
    uint32_t max_need = 0;
    uint64_t n_modal = 0, n_bool = 0;
};

void build_plan(const std::vector<Lowered> &low, const std::vector<bool> &fits, HostPlan *hp) {
    size_t longest = 1;
    for (size_t i = 0; i < low.size(); ++i)
        if (fits[i]) longest = std::max(longest, low[i].ucode.size());
    hp->stride = (uint32_t)((longest + 1 + 1) / 2 * 2);        // one spare entry after FIN (prefetch)
    for (size_t i = 0; i < low.size(); ++i) {
        if (!fits[i]) { hp->unfit.push_back((uint32_t)i); continue; }
        hp->slot_record.push_back((uint32_t)i);
        size_t at = hp->ucode.size();
        hp->ucode.resize(at + hp->stride, (uint16_t)UC_FIN_ALL);
        std::memcpy(&hp->ucode[at], low[i].ucode.data(), low[i].ucode.size() * sizeof(uint16_t));
        hp->max_need = std::max(hp->max_need, (uint32_t)low[i].need);
        hp->n_modal += low[i].n_modal;
        hp->n_bool += low[i].n_bool;
    }
}

struct DevicePlan {
    uint16_t *ucode = nullptr;
    uint32_t *slot_record = nullptr;
    uint32_t *unfit = nullptr;
    uint32_t n_slots = 0, n_unfit = 0, stride = 2, max_need = 0;
    uint64_t n_modal = 0, n_bool = 0;
    void release() {
        cudaFree(ucode); cudaFree(slot_record); cudaFree(unfit);
        ucode = nullptr; slot_record = nullptr; unfit = nullptr; n_slots = n_unfit = 0;
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
    dp->max_need = hp.max_need;
    dp->n_modal = hp.n_modal;
    dp->n_bool = hp.n_bool;
    return KRIPKE_OK;
}

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
    std::map<uint32_t, DevicePlan> single;   // one record per formula, per lowering mode (built on first use)
    DevicePlan pair;                   // rebuilt by each kripke_distinguish_pairs call
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

// The batch lowered for one set of derived leaves (cached in the handle; synchronous upload).
int single_plan(kripke_programs *h, uint32_t mode, const DevicePlan **out) {
    auto it = h->single.find(mode);
    if (it == h->single.end()) {
        std::vector<Lowered> low(h->n_formulas);
        std::vector<bool> fits(h->n_formulas);
        for (uint32_t b = 0; b < h->n_formulas; ++b)
            fits[b] = lower_single(&h->h_code[h->h_offsets[b]], h->h_offsets[b + 1] - h->h_offsets[b], mode, &low[b]);
        HostPlan hp;
        build_plan(low, fits, &hp);
        DevicePlan dp;
        int rc = upload_plan(hp, &dp);
        if (rc) { dp.release(); return rc; }
        it = h->single.emplace(mode, dp).first;
    }
    *out = &it->second;
    return KRIPKE_OK;
}

// The common scan: zero accumulators, run the sliced kernel on the aligned part of the range for
// the records it can take and the scalar kernel on the rest, then finish.
int run_scan(kripke_programs *h, const DevicePlan &plan, const uint32_t *d_pairs, uint32_t n_records,
             uint32_t n, uint32_t k, uint32_t cls, uint64_t begin, uint64_t count, uint32_t flags,
             kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream) {
    if (n < 1 || n > KRIPKE_MAX_WORLDS || k != h->n_vars || cls > KRIPKE_CLASS_S5) return KRIPKE_EINVAL;
    if (n * n + k * n > KRIPKE_MAX_MODEL_BITS) return KRIPKE_EUNSUPPORTED;
    if (flags & ~(KRIPKE_ACCUMULATE | KRIPKE_KERNEL_MASK | KRIPKE_REDUCE_MASK)) return KRIPKE_EINVAL;
    const uint32_t family = flags & KRIPKE_KERNEL_MASK, reduce = (flags & KRIPKE_REDUCE_MASK) >> 8;
    if (family == KRIPKE_KERNEL_MASK || reduce > 2) return KRIPKE_EINVAL;
    if (n_records && (!counts_out || !witness_out)) return KRIPKE_EINVAL;
    uint64_t csize = 0;
    int rc = class_size(n, cls, &csize);
    if (rc) return rc;
    if (begin > csize || count > csize - begin) return KRIPKE_EINVAL;
    h->last = kripke_run_info_t{};
    h->last.models_per_program = count << (k * n);
    h->last.sliced_logic_ops_per_word =
        plan.n_modal * n * n + plan.n_bool * n + (uint64_t)plan.n_slots * (n + 1);
    if (n_records == 0) return KRIPKE_OK;

    if ((rc = ensure_accum(h, n_records))) return rc;
    ScanJob job;
    job.n = n; job.k = k; job.cls = cls;
    job.frame_begin = begin; job.frame_count = count;
    if ((rc = class_table_device(n, cls, &job.class_table))) return rc;
    job.code = h->d_code; job.offsets = h->d_offsets; job.n_formulas = h->n_formulas;
    job.pairs = d_pairs; job.n_records = n_records;
    job.accum = h->d_accum;

    int e = launch_init(job.accum, n_records, stream);
    if (e) return cuda_fail(e);
    uint32_t launches = 1;

    // the sliced kernel runs the batch if an instantiation for this shape keeps enough stack slots
    uint64_t fpu = 1;
    bool use_sliced = family != KRIPKE_KERNEL_SCALAR && plan.n_slots > 0 &&
                      sliced_select(n, k, cls, plan.max_need, &fpu);
    uint64_t ab = begin, ae = begin;          // aligned sub-range for the sliced kernel
    if (use_sliced) {
        ab = (begin + fpu - 1) / fpu * fpu;
        ae = (begin + count) / fpu * fpu;
        if (ae <= ab) { use_sliced = false; ab = ae = begin; }
    }
    if (family == KRIPKE_KERNEL_SLICED) {
        if (!use_sliced || plan.n_unfit || ab != begin || ae != begin + count) return KRIPKE_EUNSUPPORTED;
    }
    if (use_sliced) {
        ScanJob sj = job;
        sj.frame_begin = ab; sj.frame_count = ae - ab;
        SlicedPlan sp;
        sp.ucode = plan.ucode; sp.slot_record = plan.slot_record;
        sp.n_slots = plan.n_slots; sp.stride = plan.stride; sp.max_need = plan.max_need;
        if ((e = launch_sliced(sj, sp, stream, &launches))) return cuda_fail(e);
        h->last.kernel_family = 1;
        if (plan.n_unfit && (e = launch_scalar(sj, plan.unfit, plan.n_unfit, reduce, stream, &launches)))
            return cuda_fail(e);
        ScanJob head = job, tail = job;
        head.frame_count = ab - begin;
        tail.frame_begin = ae; tail.frame_count = begin + count - ae;
        if ((e = launch_scalar(head, nullptr, n_records, reduce, stream, &launches))) return cuda_fail(e);
        if ((e = launch_scalar(tail, nullptr, n_records, reduce, stream, &launches))) return cuda_fail(e);
    } else {
        if ((e = launch_scalar(job, nullptr, n_records, reduce, stream, &launches))) return cuda_fail(e);
    }
    if ((e = launch_finish(job, (flags & KRIPKE_ACCUMULATE) != 0, counts_out, witness_out, stream)))
        return cuda_fail(e);
    h->last.launches = launches + 1;
    return KRIPKE_OK;
}

}  // namespace

extern "C" {

const char *kripke_version(void) { return "kripke-b200 0.1 (sm_100a)"; }

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
    h->n_formulas = n_formulas;
    h->n_vars = n_vars;
    h->h_offsets.assign(offsets, offsets + n_formulas + 1);
    h->h_code.assign(code + offsets[0], code + offsets[n_formulas]);
    const uint32_t base = offsets[0];
    for (auto &o : h->h_offsets) o -= base;
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
    cudaDeviceSynchronize();
    for (auto &kv : h->single) kv.second.release();
    h->pair.release();
    cudaFree(h->d_code); cudaFree(h->d_offsets); cudaFree(h->d_pairs); cudaFree(h->d_accum);
    cudaFree(h->d_tmp_counts); cudaFree(h->d_tmp_wit);
    delete h;
    return KRIPKE_OK;
}

int kripke_eval_batch_range(const kripke_programs_t *programs, uint32_t n_worlds, uint32_t n_vars,
                            uint32_t frame_class, uint64_t frame_begin, uint64_t frame_count,
                            uint32_t flags, kripke_count_t *counts_out, kripke_witness_t *witness_out,
                            void *stream) {
    if (!programs) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    const DevicePlan *plan = nullptr;
    int rc = single_plan(h, sliced_lower_mode(n_worlds, n_vars), &plan);
    if (rc) return rc;
    return run_scan(h, *plan, nullptr, h->n_formulas, n_worlds, n_vars, frame_class, frame_begin,
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
    const uint32_t mode = sliced_lower_mode(n_worlds, n_vars);
    std::vector<Lowered> low(n_pairs);
    std::vector<bool> fits(n_pairs);
    for (uint32_t j = 0; j < n_pairs; ++j) {
        const uint32_t a = pairs[2 * j], b = pairs[2 * j + 1];
        fits[j] = lower_pair(&h->h_code[h->h_offsets[a]], h->h_offsets[a + 1] - h->h_offsets[a],
                             &h->h_code[h->h_offsets[b]], h->h_offsets[b + 1] - h->h_offsets[b], mode, &low[j]);
    }
    HostPlan hp;
    build_plan(low, fits, &hp);
    // the previous call's plan may still be in use on another stream: wait before replacing it
    CU(cudaDeviceSynchronize());
    int rc = upload_plan(hp, &h->pair);
    if (rc) return rc;
    if (n_pairs > h->pairs_cap) {
        cudaFree(h->d_pairs);
        h->d_pairs = nullptr; h->pairs_cap = 0;
        CU(cudaMalloc((void **)&h->d_pairs, (size_t)2 * n_pairs * sizeof(uint32_t)));
        h->pairs_cap = n_pairs;
    }
    if (n_pairs) CU(cudaMemcpy(h->d_pairs, pairs, (size_t)2 * n_pairs * sizeof(uint32_t), cudaMemcpyHostToDevice));
    return run_scan(h, h->pair, h->d_pairs, n_pairs, n_worlds, n_vars, frame_class, frame_begin,
                    frame_count, flags, counts_out, witness_out, stream);
}

int kripke_minimal_refutation(const kripke_programs_t *programs, uint32_t n_vars, uint32_t frame_class,
                              uint32_t n_max, uint32_t *size_out, kripke_count_t *counts_out,
                              kripke_witness_t *witness_out, void *stream) {
    if (!programs || n_max < 1 || n_max > KRIPKE_MAX_WORLDS) return KRIPKE_EINVAL;
    kripke_programs *h = const_cast<kripke_programs *>(programs);
    const uint32_t B = h->n_formulas;
    if (B && (!size_out || !counts_out || !witness_out)) return KRIPKE_EINVAL;
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
    std::vector<uint32_t> sub;
    int rc = KRIPKE_OK;
    for (uint32_t n = 1; n <= n_max && rc == KRIPKE_OK && !active.empty(); ++n) {
        const uint64_t total = 1ull << (n * n);
        for (uint64_t begin = 0; begin < total && rc == KRIPKE_OK && !active.empty(); begin += chunk_frames) {
            const uint64_t count = std::min<uint64_t>(chunk_frames, total - begin);
            sub.resize(2 * active.size());
            for (size_t a = 0; a < active.size(); ++a) {
                sub[2 * a] = pairs[2 * active[a]];
                sub[2 * a + 1] = pairs[2 * active[a] + 1];
            }
            rc = kripke_distinguish_pairs(h, sub.data(), (uint32_t)active.size(), n, n_vars, KRIPKE_CLASS_K, begin,
                                          count, 0, d_counts, d_wit, stream);
            if (rc) break;
            cudaError_t e = cudaMemcpyAsync(hc.data(), d_counts, active.size() * sizeof(kripke_count_t),
                                            cudaMemcpyDeviceToHost, (cudaStream_t)stream);
            if (e == cudaSuccess)
                e = cudaMemcpyAsync(hw.data(), d_wit, active.size() * sizeof(kripke_witness_t),
                                    cudaMemcpyDeviceToHost, (cudaStream_t)stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
            if (e != cudaSuccess) { rc = cuda_fail((int)e); break; }
            std::vector<uint32_t> still;
            for (size_t a = 0; a < active.size(); ++a) {
                if (hc[a].refuting_models != 0) {
                    size_out[active[a]] = n;
                    witness_out[active[a]] = hw[a];
                } else {
                    still.push_back(active[a]);
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
    if (leaf_mode > 3) return KRIPKE_EINVAL;
    const bool fits = code_b ? lower_pair(code_a, len_a, code_b, len_b, leaf_mode, &low)
                             : lower_single(code_a, len_a, leaf_mode, &low);
    if (need_out) *need_out = (uint32_t)low.need;
    if (!fits) return KRIPKE_EUNSUPPORTED;
    if (low.ucode.size() > cap) return KRIPKE_EINVAL;
    std::memcpy(ucode_out, low.ucode.data(), low.ucode.size() * sizeof(uint16_t));
    return (int)low.ucode.size();
}

int kripke_calibrate_int32(uint32_t variant, double *thread_instr_per_s_out, double *elapsed_ms_out,
                           void *stream) {
    if (variant > 3 || !thread_instr_per_s_out) return KRIPKE_EINVAL;
    int e = run_calibration(variant, thread_instr_per_s_out, elapsed_ms_out, stream);
    if (e) return cuda_fail(e);
    return KRIPKE_OK;
}

}  // extern "C"
