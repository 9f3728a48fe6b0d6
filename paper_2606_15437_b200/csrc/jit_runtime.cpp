// jit_runtime.cpp - NVRTC compilation, the per-process module cache and the launches of the compiled
// scans (jit.h).  Kernels are compiled for sm_100a only (--gpu-architecture=sm_100a, straight to SASS:
// no PTX is kept and nothing is JIT-compiled by the driver).
#include <cuda_runtime.h>
#include <nvrtc.h>

#include <algorithm>
#include <atomic>
#include <map>
#include <mutex>
#include <thread>

#include "jit.h"

namespace kripke {

namespace {

// must match KjParams in jit_prelude.inc
struct KjParamsHost {
    unsigned long long unit_begin, unit_count;
    const unsigned long long *class_table;
    const unsigned *slot_record;
    Accum *accum;
    unsigned units_per_item, n_items;
    unsigned model_shift, pad;
    unsigned *density;
    unsigned long long total_frames, frame_base;
    const unsigned *row_begin, *rows;
};

struct Module {
    cudaLibrary_t lib = nullptr;
    cudaKernel_t kernel = nullptr;
    int regs = 0;
    int local_bytes = 0;       // per-thread local memory: nonzero = ptxas spilled registers
};

std::mutex g_cache_mutex;
// source text -> loaded module.  Modules stay loaded until jit_cache_clear(): plans hold their kernel handles.
std::map<std::string, Module> g_cache;

int compile(const std::string &src, std::vector<char> *cubin, std::string *log) {
    nvrtcProgram prog = nullptr;
    if (nvrtcCreateProgram(&prog, src.c_str(), "kripke_jit.cu", 0, nullptr, nullptr) != NVRTC_SUCCESS) return KRIPKE_ENOMEM;
    const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo"};
    const nvrtcResult r = nvrtcCompileProgram(prog, 3, opts);
    if (r != NVRTC_SUCCESS) {
        if (log) {
            size_t n = 0;
            nvrtcGetProgramLogSize(prog, &n);
            log->resize(n);
            if (n) nvrtcGetProgramLog(prog, &(*log)[0]);
        }
        nvrtcDestroyProgram(&prog);
        return KRIPKE_EUNSUPPORTED;
    }
    size_t n = 0;
    nvrtcGetCUBINSize(prog, &n);
    cubin->resize(n);
    nvrtcGetCUBIN(prog, cubin->data());
    nvrtcDestroyProgram(&prog);
    return n ? 0 : KRIPKE_EUNSUPPORTED;
}

}  // namespace

void JitGroupPlan::release() {
    cudaFree(d_slot_record);
    cudaFree(d_row_begin);
    cudaFree(d_rows);
    d_slot_record = d_row_begin = d_rows = nullptr;
    kernels.clear();
    n_slots = 0;
}

size_t jit_cache_clear() {
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    const size_t n = g_cache.size();
    for (auto &kv : g_cache)
        if (kv.second.lib) cudaLibraryUnload(kv.second.lib);
    g_cache.clear();
    return n;
}

size_t jit_cache_modules() {
    std::lock_guard<std::mutex> lock(g_cache_mutex);
    return g_cache.size();
}

int jit_compile_only(const std::string &source, std::string *log_out, size_t *cubin_bytes) {
    std::vector<char> cubin;
    const int rc = compile(source, &cubin, log_out);
    if (cubin_bytes) *cubin_bytes = cubin.size();
    return rc;
}

int jit_build_group(const Dag &dag, const JitLayout &lay, const std::vector<JitRoot> &roots,
                    const std::vector<uint32_t> &slot_record, uint32_t max_roots, uint32_t min_blocks,
                    uint32_t mode, JitGroupPlan *out, std::string *log_out) {
    out->release();
    out->lay = lay;
    out->stats = JitEmitStats();
    out->threads = 128;
    if (roots.empty()) return 0;
    std::vector<std::vector<uint32_t>> parts;
    if (mode == JIT_MODE_DENSITY) {
        // every record writes its own row: records in order, max_roots per kernel (the graph is still shared)
        for (uint32_t r = 0; r < roots.size(); ++r) {
            if (r % max_roots == 0) parts.emplace_back();
            parts.back().push_back(r);
        }
    } else {
        parts = jit_partition(dag, roots, lay, max_roots);
    }
    // Emit, compile (what the process has not seen yet, in parallel host threads) and load; a kernel that ptxas
    // could only fit by spilling registers to local memory is split into two halves and redone.
    std::vector<std::string> sources;
    std::vector<JitEmitStats> stats;
    for (int round = 0;; ++round) {
        sources.assign(parts.size(), std::string());
        stats.assign(parts.size(), JitEmitStats());
        for (size_t i = 0; i < parts.size(); ++i) {
            std::vector<JitRoot> rs;
            for (uint32_t r : parts[i]) rs.push_back(roots[r]);
            sources[i] = jit_emit_kernel(dag, lay, rs, out->threads, min_blocks, mode, &stats[i]);
        }
        std::vector<size_t> todo;
        {
            std::lock_guard<std::mutex> lock(g_cache_mutex);
            for (size_t i = 0; i < sources.size(); ++i)
                if (!g_cache.count(sources[i]) &&
                    std::find_if(todo.begin(), todo.end(), [&](size_t j) { return sources[j] == sources[i]; }) == todo.end())
                    todo.push_back(i);
        }
        std::vector<std::vector<char>> cubins(todo.size());
        std::vector<int> rcs(todo.size(), 0);
        std::vector<std::string> logs(todo.size());
        {
            std::atomic<size_t> next{0};
            const unsigned hw = std::max(1u, std::thread::hardware_concurrency());
            const size_t n_threads = std::min<size_t>(todo.size(), hw);
            std::vector<std::thread> pool;
            auto work = [&]() {
                for (size_t t = next++; t < todo.size(); t = next++) rcs[t] = compile(sources[todo[t]], &cubins[t], &logs[t]);
            };
            for (size_t t = 1; t < n_threads; ++t) pool.emplace_back(work);
            if (n_threads) work();
            for (auto &th : pool) th.join();
        }
        for (size_t t = 0; t < todo.size(); ++t)
            if (rcs[t]) {
                if (log_out) *log_out = logs[t];
                return rcs[t];
            }
        bool split = false;
        {
            std::lock_guard<std::mutex> lock(g_cache_mutex);
            for (size_t t = 0; t < todo.size(); ++t) {
                // another thread may have compiled and loaded the same source since `todo` was made: keep its module
                if (g_cache.count(sources[todo[t]])) continue;
                Module m;
                cudaError_t e = cudaLibraryLoadData(&m.lib, cubins[t].data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
                if (e == cudaSuccess) e = cudaLibraryGetKernel(&m.kernel, m.lib, "kripke_jit_scan");
                cudaFuncAttributes attr;
                if (e == cudaSuccess) e = cudaFuncGetAttributes(&attr, (const void *)m.kernel);
                if (e != cudaSuccess) {
                    if (m.lib) cudaLibraryUnload(m.lib);
                    return (int)e;
                }
                m.regs = attr.numRegs;
                m.local_bytes = (int)attr.localSizeBytes;
                g_cache.emplace(sources[todo[t]], m);
            }
            if (mode != JIT_MODE_DENSITY && round < 4) {
                std::vector<std::vector<uint32_t>> next_parts;
                for (size_t i = 0; i < parts.size(); ++i) {
                    if (g_cache[sources[i]].local_bytes > 0 && parts[i].size() >= 16) {
                        // its programs are partitioned again, into two kernels with about the same work
                        std::vector<JitRoot> sub;
                        for (uint32_t r : parts[i]) sub.push_back(roots[r]);
                        for (const auto &sp : jit_partition(dag, sub, lay, (uint32_t)(parts[i].size() + 1) / 2)) {
                            next_parts.emplace_back();
                            for (uint32_t j : sp) next_parts.back().push_back(parts[i][j]);
                        }
                        split = true;
                    } else {
                        next_parts.push_back(parts[i]);
                    }
                }
                if (split) parts.swap(next_parts);
            }
        }
        if (!split) break;
    }
    std::vector<uint32_t> order;               // slot -> index into roots
    {
        std::lock_guard<std::mutex> lock(g_cache_mutex);
        uint32_t base = 0;
        for (size_t i = 0; i < parts.size(); ++i) {
            for (uint32_t r : parts[i]) order.push_back(r);
            out->stats.logic_ops_per_word += stats[i].logic_ops_per_word;
            out->stats.logic_ops_emitted += stats[i].logic_ops_emitted;
            out->stats.n_box += stats[i].n_box;
            out->stats.n_and += stats[i].n_and;
            JitKernel k;
            k.kernel = (void *)g_cache[sources[i]].kernel;
            k.slot_base = base;
            k.n_slots = (uint32_t)parts[i].size();
            base += k.n_slots;
            out->kernels.push_back(k);
        }
    }
    out->h_slot_record.resize(order.size());
    for (size_t s = 0; s < order.size(); ++s) out->h_slot_record[s] = slot_record[order[s]];
    return jit_upload_slots(out);
}

int jit_upload_slots(JitGroupPlan *plan) {
    const std::vector<uint32_t> &records = plan->h_slot_record;
    plan->n_slots = (uint32_t)records.size();
    if (records.empty()) return 0;
    auto up = [](uint32_t **dst, const std::vector<uint32_t> &src) {
        cudaFree(*dst);
        *dst = nullptr;
        if (src.empty()) return cudaSuccess;
        cudaError_t e = cudaMalloc((void **)dst, src.size() * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMemcpy(*dst, src.data(), src.size() * sizeof(uint32_t), cudaMemcpyHostToDevice);
        return e;
    };
    cudaError_t e = up(&plan->d_slot_record, records);
    if (e == cudaSuccess) e = up(&plan->d_row_begin, plan->h_row_begin);
    if (e == cudaSuccess) e = up(&plan->d_rows, plan->h_rows);
    return (int)e;
}

int jit_launch_group(const ScanJob &job, const JitGroupPlan &plan, uint32_t model_shift, const JitDensityOut *density,
                     void *stream, uint32_t *launches) {
    const JitLayout &lay = plan.lay;
    if (job.frame_count == 0 || plan.kernels.empty()) return 0;
    int dev = 0, sm_count = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    // frames -> units: 2^split units per frame, or 2^unit_frames_log2 frames per unit (the caller aligned the range)
    KjParamsHost p;
    p.unit_begin = (job.frame_begin >> lay.unit_frames_log2) << lay.split;
    p.unit_count = (job.frame_count >> lay.unit_frames_log2) << lay.split;
    p.class_table = (const unsigned long long *)job.class_table;
    p.accum = job.accum;
    p.model_shift = model_shift;
    p.pad = 0;
    p.density = density ? density->counts : nullptr;
    p.total_frames = density ? density->total_frames : 0;
    p.frame_base = density ? density->frame_base : 0;
    p.row_begin = nullptr;
    p.rows = nullptr;
    if (p.unit_count == 0) return 0;
    const uint32_t threads = plan.threads;
    const uint64_t tiles = (p.unit_count + threads - 1) / threads;
    // a block's per-item model count is a 32-bit shared-memory counter: bound the item
    const uint32_t unit_models_log2 = 5 + lay.inner + lay.outer;
    const uint64_t max_tiles_per_item = std::max<uint64_t>(1, (1ull << (31 - unit_models_log2)) / threads);
    for (const JitKernel &k : plan.kernels) {
        cudaFuncAttributes attr;
        if ((e = cudaFuncGetAttributes(&attr, (const void *)k.kernel)) != cudaSuccess) return (int)e;
        const int regs = std::max(32, (attr.numRegs + 7) / 8 * 8);
        const uint32_t blocks_per_sm = (uint32_t)std::max(1, std::min(16, 65536 / (regs * (int)threads)));
        const uint64_t grid_full = (uint64_t)sm_count * blocks_per_sm;
        uint64_t tiles_per_item = std::max<uint64_t>(1, std::min<uint64_t>(64, tiles / (grid_full * 16)));
        tiles_per_item = std::min(tiles_per_item, max_tiles_per_item);
        const uint64_t n_items = (tiles + tiles_per_item - 1) / tiles_per_item;
        const uint64_t max_items = 0x7FFFFFFFull;
        for (uint64_t i0 = 0; i0 < n_items; i0 += max_items) {
            KjParamsHost q = p;
            const uint64_t ni = std::min(max_items, n_items - i0);
            q.units_per_item = (unsigned)(tiles_per_item * threads);
            q.unit_begin = p.unit_begin + i0 * q.units_per_item;
            q.unit_count = std::min<uint64_t>(p.unit_count - i0 * q.units_per_item, ni * q.units_per_item);
            q.n_items = (unsigned)ni;
            q.slot_record = plan.d_slot_record + k.slot_base;
            q.row_begin = plan.d_row_begin ? plan.d_row_begin + k.slot_base : nullptr;
            q.rows = plan.d_rows;
            void *args[] = {&q};
            const unsigned grid = (unsigned)std::min<uint64_t>(ni, grid_full);
            e = cudaLaunchKernel((const void *)k.kernel, dim3(grid), dim3(threads), args, 0, (cudaStream_t)stream);
            if (e != cudaSuccess) return (int)e;
            if (launches) ++*launches;
        }
    }
    return 0;
}

}  // namespace kripke
