// scan_scalar.cu - the scalar scan (Algorithm 1 restated), accumulator init and the
// witness-completion ("finish") kernel.
//
// The scalar kernel is the paper's own layout: thread = frame, loop over formulas, loop over
// valuations, one model per iteration on n-bit masks, hierarchical reduction.  In this
// library it is the general fallback (any n <= 6, any class, any range, programs too deep for the
// register stack of the bit-sliced kernel), the cross-check of the bit-sliced kernel, and the
// baseline of the layout / atomic-contention ablations.  The hot path is
// scan_sliced.cuh.
#include <cuda_runtime.h>

#include <algorithm>

#include "frames.cuh"
#include "internal.h"

namespace kripke {

namespace {

constexpr int SCALAR_THREADS = 256;

struct ScalarParams {
    uint32_t n, k, cls;
    uint64_t frame_begin, frame_end;      // class-order range
    const uint64_t *class_table;
    const uint8_t *code;
    const uint32_t *offsets;
    const uint32_t *pairs;                // null = one record per formula
    const uint32_t *records;              // null = records 0..n_list-1
    uint32_t n_list;
    uint32_t chunk;                       // records per blockIdx.y
    uint32_t reduce_mode;                 // 0 block, 1 warp, 2 thread
    Accum *accum;
};

__device__ __forceinline__ void decode_succ(uint32_t n, uint64_t f, uint32_t *succ) {
    const uint32_t full = (1u << n) - 1u;
    for (uint32_t w = 0; w < KRIPKE_MAX_WORLDS; ++w) succ[w] = (w < n) ? (uint32_t)(f >> (w * n)) & full : 0u;
}

__global__ void __launch_bounds__(SCALAR_THREADS) scan_scalar_kernel(ScalarParams p) {
    __shared__ unsigned long long s_models[SCALAR_THREADS / 32];
    __shared__ uint32_t s_frames[SCALAR_THREADS / 32];
    __shared__ unsigned long long s_best[SCALAR_THREADS / 32];

    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint64_t c = p.frame_begin + (uint64_t)blockIdx.x * SCALAR_THREADS + threadIdx.x;   // class-order index
    const bool valid = c < p.frame_end;
    const uint32_t full = (1u << p.n) - 1u;
    uint32_t succ[KRIPKE_MAX_WORLDS];
    decode_succ(p.n, valid ? class_frame(p.n, p.cls, p.class_table, c) : 0ull, succ);   // step H2
    const uint64_t nval = 1ull << (p.k * p.n);

    const uint32_t r0 = blockIdx.y * p.chunk;
    const uint32_t r1 = min(r0 + p.chunk, p.n_list);
    for (uint32_t li = r0; li < r1; ++li) {
        const uint32_t rec = p.records ? p.records[li] : li;
        const uint32_t fa = p.pairs ? p.pairs[2 * rec] : rec;
        const uint32_t fb = p.pairs ? p.pairs[2 * rec + 1] : rec;
        const uint8_t *ca = p.code + p.offsets[fa];
        const uint32_t la = p.offsets[fa + 1] - p.offsets[fa];
        const uint8_t *cb = p.code + p.offsets[fb];
        const uint32_t lb = p.offsets[fb + 1] - p.offsets[fb];
        unsigned long long lf = 0;                       // Algorithm 1 line 5
        if (valid) {
            for (uint64_t v = 0; v < nval; ++v) {        // line 6; step H3: masks from the index
                uint32_t val[KRIPKE_MAX_VARS];
                for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) val[i] = (uint32_t)(v >> (i * p.n)) & full;
                const uint32_t t = eval_postfix_scalar(ca, la, p.n, succ, val, full);   // line 7
                bool hit;
                if (p.pairs) hit = (t ^ eval_postfix_scalar(cb, lb, p.n, succ, val, full)) != 0u;
                else hit = t != full;                    // line 8
                lf += hit;
            }
        }
        // step H6: hierarchical reduction
        if (p.reduce_mode == 2) {                        // frame atomics (the paper's first version)
            if (lf) {
                atomicAdd(&p.accum[rec].models, lf);
                atomicAdd(&p.accum[rec].frames, 1ull);
                atomicMin(&p.accum[rec].best, (unsigned long long)c);
            }
            continue;
        }
        const uint32_t bal = __ballot_sync(0xffffffffu, lf != 0);
        unsigned long long wsum = lf;
        for (int o = 16; o > 0; o >>= 1) wsum += __shfl_xor_sync(0xffffffffu, wsum, o);
        const unsigned long long wbest = bal ? (c - lane + (__ffs(bal) - 1)) : ~0ull;
        if (p.reduce_mode == 1) {
            if (lane == 0 && bal) {
                atomicAdd(&p.accum[rec].models, wsum);
                atomicAdd(&p.accum[rec].frames, (unsigned long long)__popc(bal));
                atomicMin(&p.accum[rec].best, wbest);
            }
            continue;
        }
        if (lane == 0) { s_models[warp] = wsum; s_frames[warp] = __popc(bal); s_best[warp] = wbest; }
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long m = 0, best = ~0ull;
            uint32_t fr = 0;
            for (int i = 0; i < SCALAR_THREADS / 32; ++i) {
                m += s_models[i]; fr += s_frames[i]; best = min(best, s_best[i]);
            }
            if (fr) {                                    // at most one atomic triple per (block, formula)
                atomicAdd(&p.accum[rec].models, m);
                atomicAdd(&p.accum[rec].frames, (unsigned long long)fr);
                atomicMin(&p.accum[rec].best, best);
            }
        }
        __syncthreads();
    }
}

__global__ void init_accum_kernel(Accum *accum, uint32_t n) {
    uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { accum[i].models = 0; accum[i].frames = 0; accum[i].best = ~0ull; }
}

struct FinishParams {
    uint32_t n, k, cls;
    uint64_t frame_end;
    const uint64_t *class_table;
    const uint8_t *code;
    const uint32_t *offsets;
    const uint32_t *pairs;
    uint32_t n_records;
    const Accum *accum;
    int accumulate;
    kripke_count_t *counts;
    kripke_witness_t *witness;
};

// One warp per record.  accum.best is a lower bound (class-order index) of the first refuting frame
// with a hit guaranteed at or shortly after it; lanes scan the models (frame, valuation) from there
// in ascending order, 32 at a time, with the scalar recurrence, and the first hit is the
// lexicographically first countermodel (step H5/H6 witness; reading R7).
__global__ void __launch_bounds__(128) finish_kernel(FinishParams p) {
    const uint32_t rec = blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5);
    const uint32_t lane = threadIdx.x & 31u;
    if (rec >= p.n_records) return;
    const Accum a = p.accum[rec];
    uint64_t wf = KRIPKE_NO_WITNESS;
    uint32_t wv = 0, ww = 0;
    if (a.best != ~0ull) {
        const uint32_t fa = p.pairs ? p.pairs[2 * rec] : rec;
        const uint32_t fb = p.pairs ? p.pairs[2 * rec + 1] : rec;
        const uint8_t *ca = p.code + p.offsets[fa];
        const uint32_t la = p.offsets[fa + 1] - p.offsets[fa];
        const uint8_t *cb = p.code + p.offsets[fb];
        const uint32_t lb = p.offsets[fb + 1] - p.offsets[fb];
        const uint32_t full = (1u << p.n) - 1u;
        const uint32_t kn = p.k * p.n;
        const uint64_t vmask = (1ull << kn) - 1ull;
        const uint64_t limit = (p.frame_end - a.best) << kn;     // models available from a.best on
        for (uint64_t base = 0; base < limit; base += 32) {
            const uint64_t x = base + lane;
            uint32_t fail = 0;
            uint64_t f = 0;
            if (x < limit) {
                const uint64_t c = a.best + (x >> kn);
                const uint64_t v = x & vmask;
                f = class_frame(p.n, p.cls, p.class_table, c);
                uint32_t succ[KRIPKE_MAX_WORLDS], val[KRIPKE_MAX_VARS];
                decode_succ(p.n, f, succ);
                for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) val[i] = (uint32_t)(v >> (i * p.n)) & full;
                const uint32_t t = eval_postfix_scalar(ca, la, p.n, succ, val, full);
                if (p.pairs) fail = t ^ eval_postfix_scalar(cb, lb, p.n, succ, val, full);
                else fail = full & ~t;
            }
            const uint32_t bal = __ballot_sync(0xffffffffu, fail != 0u);
            if (bal) {
                const int src = __ffs(bal) - 1;
                wf = __shfl_sync(0xffffffffu, f, src);
                wv = (uint32_t)(__shfl_sync(0xffffffffu, x, src) & vmask);
                ww = __ffs(__shfl_sync(0xffffffffu, fail, src)) - 1;
                break;
            }
        }
    }
    if (lane == 0) {
        kripke_count_t cnt;
        cnt.refuting_models = a.models;
        cnt.refuting_frames = a.frames;
        kripke_witness_t wit;
        wit.frame = wf; wit.valuation = wv; wit.world = ww;
        if (p.accumulate) {
            const kripke_count_t oc = p.counts[rec];
            const kripke_witness_t ow = p.witness[rec];
            cnt.refuting_models += oc.refuting_models;
            cnt.refuting_frames += oc.refuting_frames;
            const bool keep_old = ow.frame != KRIPKE_NO_WITNESS &&
                                  (wf == KRIPKE_NO_WITNESS || ow.frame < wf || (ow.frame == wf && ow.valuation <= wv));
            if (keep_old) wit = ow;
        }
        p.counts[rec] = cnt;
        p.witness[rec] = wit;
    }
}

__global__ void witness_to_keys_kernel(const kripke_witness_t *wit, uint32_t n, uint32_t kn, unsigned long long *keys) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const kripke_witness_t w = wit[i];
    keys[i] = (w.frame == KRIPKE_NO_WITNESS) ? 0x7FFFFFFFFFFFFFFFull
                                             : ((((w.frame << kn) | w.valuation) << 3) | w.world);
}

__global__ void keys_to_witness_kernel(const unsigned long long *keys, uint32_t n, uint32_t kn, kripke_witness_t *wit) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const unsigned long long key = keys[i];
    kripke_witness_t w;
    if (key == 0x7FFFFFFFFFFFFFFFull) { w.frame = KRIPKE_NO_WITNESS; w.valuation = 0; w.world = 0; }
    else {
        w.world = (uint32_t)(key & 7ull);
        w.valuation = (uint32_t)((key >> 3) & ((1ull << kn) - 1ull));
        w.frame = key >> (kn + 3);
    }
    wit[i] = w;
}

// step H8: keep the first size at which a formula is refuted
__global__ void record_size_kernel(uint32_t n, uint32_t n_records, const kripke_count_t *cnt, const kripke_witness_t *wit,
                                   uint32_t *size_out, kripke_count_t *counts_out, kripke_witness_t *witness_out) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_records) return;
    if (n == 1) {
        size_out[i] = 0;
        counts_out[i].refuting_models = 0; counts_out[i].refuting_frames = 0;
        witness_out[i].frame = KRIPKE_NO_WITNESS; witness_out[i].valuation = 0; witness_out[i].world = 0;
    }
    if (size_out[i] == 0 && cnt[i].refuting_models != 0) {
        size_out[i] = n;
        counts_out[i] = cnt[i];
        witness_out[i] = wit[i];
    }
}

}  // namespace

int launch_record_size(uint32_t n, uint32_t n_records, const kripke_count_t *cnt, const kripke_witness_t *wit,
                       uint32_t *size_out, kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream) {
    if (n_records == 0) return 0;
    record_size_kernel<<<(n_records + 255) / 256, 256, 0, (cudaStream_t)stream>>>(n, n_records, cnt, wit, size_out,
                                                                                  counts_out, witness_out);
    return (int)cudaGetLastError();
}

int launch_witness_keys(bool to_keys, const void *src, uint32_t n_records, uint32_t kn, void *dst, void *stream) {
    if (n_records == 0) return 0;
    const uint32_t grid = (n_records + 255) / 256;
    if (to_keys)
        witness_to_keys_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((const kripke_witness_t *)src, n_records, kn,
                                                                       (unsigned long long *)dst);
    else
        keys_to_witness_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>((const unsigned long long *)src, n_records, kn,
                                                                       (kripke_witness_t *)dst);
    return (int)cudaGetLastError();
}

int launch_scalar(const ScanJob &job, const uint32_t *records, uint32_t n_list, uint32_t reduce_mode,
                  void *stream, uint32_t *launches) {
    if (n_list == 0 || job.frame_count == 0) return 0;
    ScalarParams p;
    p.n = job.n; p.k = job.k; p.cls = job.cls;
    p.frame_begin = job.frame_begin; p.frame_end = job.frame_begin + job.frame_count;
    p.class_table = job.class_table;
    p.code = job.code; p.offsets = job.offsets; p.pairs = job.pairs;
    p.records = records; p.n_list = n_list;
    p.reduce_mode = reduce_mode;
    p.accum = job.accum;
    // Parallelism over frames (as in the paper) and, when frames are few, over record chunks too
    // (the paper's kernel underfills on small filtered classes).
    const uint64_t tiles = (job.frame_count + SCALAR_THREADS - 1) / SCALAR_THREADS;
    const uint64_t max_tiles_per_launch = 1u << 30;
    uint32_t chunks = 1;
    if (tiles < 2048) {
        uint64_t want = (2048 + tiles - 1) / tiles;
        chunks = (uint32_t)std::min<uint64_t>(want, n_list);
    }
    chunks = std::min<uint32_t>(chunks, 65535u);
    p.chunk = (n_list + chunks - 1) / chunks;
    const uint32_t grid_y = (n_list + p.chunk - 1) / p.chunk;
    for (uint64_t t0 = 0; t0 < tiles; t0 += max_tiles_per_launch) {
        const uint64_t nt = std::min<uint64_t>(max_tiles_per_launch, tiles - t0);
        ScalarParams q = p;
        q.frame_begin = p.frame_begin + t0 * SCALAR_THREADS;
        scan_scalar_kernel<<<dim3((unsigned)nt, grid_y), SCALAR_THREADS, 0, (cudaStream_t)stream>>>(q);
        if (launches) ++*launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return (int)e;
    }
    return 0;
}

__global__ void alias_accum_kernel(Accum *accum, const uint32_t *pairs, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) accum[pairs[2 * i]] = accum[pairs[2 * i + 1]];
}

int launch_alias_accum(Accum *accum, const uint32_t *pairs, uint32_t n, void *stream) {
    if (n == 0) return 0;
    alias_accum_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>(accum, pairs, n);
    return (int)cudaGetLastError();
}

int launch_init(Accum *accum, uint32_t n_records, void *stream) {
    if (n_records == 0) return 0;
    init_accum_kernel<<<(n_records + 255) / 256, 256, 0, (cudaStream_t)stream>>>(accum, n_records);
    return (int)cudaGetLastError();
}

int launch_finish(const ScanJob &job, bool accumulate, kripke_count_t *counts_out,
                  kripke_witness_t *witness_out, void *stream) {
    if (job.n_records == 0) return 0;
    FinishParams p;
    p.n = job.n; p.k = job.k; p.cls = job.cls;
    p.frame_end = job.frame_begin + job.frame_count;
    p.class_table = job.class_table;
    p.code = job.code; p.offsets = job.offsets; p.pairs = job.pairs;
    p.n_records = job.n_records;
    p.accum = job.accum;
    p.accumulate = accumulate ? 1 : 0;
    p.counts = counts_out; p.witness = witness_out;
    finish_kernel<<<(job.n_records + 3) / 4, 128, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

}  // namespace kripke
