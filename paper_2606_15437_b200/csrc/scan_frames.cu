// scan_frames.cu - frame-list mode: dispatch over the bit-sliced instantiations
// (scan_frames.cuh, scan_frames_inst.cu), the scalar kernel and the witness-completion kernel.
#include <cuda_runtime.h>

#include <algorithm>

#include "frames.cuh"
#include "internal.h"

namespace kripke {

// scan_frames_inst.cu: launch_frames_<N>_v<VB>
#define FR_DECL(N) \
    int launch_frames_##N##_v1(const FramesJob &, const SlicedPlan &, void *, uint32_t *); \
    int launch_frames_##N##_v2(const FramesJob &, const SlicedPlan &, void *, uint32_t *); \
    int launch_frames_##N##_v4(const FramesJob &, const SlicedPlan &, void *, uint32_t *);
FR_DECL(1) FR_DECL(2) FR_DECL(3) FR_DECL(4) FR_DECL(5) FR_DECL(6) FR_DECL(7) FR_DECL(8)
FR_DECL(9) FR_DECL(10) FR_DECL(11) FR_DECL(12) FR_DECL(13) FR_DECL(14) FR_DECL(15) FR_DECL(16)
#undef FR_DECL

namespace {

// Scalar form (the paper's own layout, Algorithm 1: thread = frame, one model per iteration on
// n-bit masks): records whose programs need more register-stack slots than the lowering keeps, the
// KRIPKE_KERNEL_SCALAR cross-check and the layout ablation.
struct FramesScalarParams {
    const uint16_t *succ;
    uint64_t n_frames;
    uint32_t n, k;
    const uint8_t *code;
    const uint32_t *offsets;
    const uint32_t *pairs;
    const uint32_t *records;       // list of record indices, or null = 0..n_list-1
    uint32_t n_list;
    Accum *accum;
};

__global__ void __launch_bounds__(128) scan_frames_scalar_kernel(FramesScalarParams p) {
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t full = (1u << p.n) - 1u;
    const uint64_t nval = 1ull << (p.k * p.n);
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    const uint64_t rounds = (p.n_frames + stride - 1) / stride;
    for (uint64_t it = 0; it < rounds; ++it) {
        const uint64_t j = it * stride + (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
        const bool valid = j < p.n_frames;
        uint32_t succ[KRIPKE_LIST_MAX_WORLDS];
        for (uint32_t w = 0; w < p.n; ++w) succ[w] = valid ? (uint32_t)p.succ[j * p.n + w] : 0u;
        for (uint32_t q = 0; q < p.n_list; ++q) {
            const uint32_t rec = p.records ? p.records[q] : q;
            const uint32_t fa = p.pairs ? p.pairs[2 * rec] : rec, fb = p.pairs ? p.pairs[2 * rec + 1] : rec;
            const uint8_t *ca = p.code + p.offsets[fa], *cb = p.code + p.offsets[fb];
            const uint32_t la = p.offsets[fa + 1] - p.offsets[fa], lb = p.offsets[fb + 1] - p.offsets[fb];
            uint32_t cnt = 0;
            if (valid) {
                for (uint64_t v = 0; v < nval; ++v) {
                    uint32_t val[KRIPKE_MAX_VARS];
                    for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) val[i] = (uint32_t)(v >> (i * p.n)) & full;
                    const uint32_t t = eval_postfix_scalar(ca, la, p.n, succ, val, full);
                    const uint32_t fail = p.pairs ? (t ^ eval_postfix_scalar(cb, lb, p.n, succ, val, full)) : (full & ~t);
                    cnt += fail != 0u;
                }
            }
            const uint32_t bal = __ballot_sync(0xFFFFFFFFu, cnt != 0u);
            if (bal) {
                const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, cnt);
                if (lane == 0) {
                    Accum *a = p.accum + rec;
                    atomicAdd(&a->models, (unsigned long long)tot);
                    atomicAdd(&a->frames, (unsigned long long)__popc(bal));
                    atomicMin(&a->best, (j - lane) + (uint64_t)(__ffs(bal) - 1));
                }
            }
        }
    }
}

// Accumulators -> counts and certificates: the first refuting (position, valuation) of the least
// refuting list position found by the scan, and its least failing world.
struct FramesFinishParams {
    const uint16_t *succ;
    uint32_t n, k;
    const uint8_t *code;
    const uint32_t *offsets;
    const uint32_t *pairs;
    uint32_t n_records;
    const Accum *accum;
    uint64_t index_base;
    bool accumulate;
    kripke_count_t *counts;
    kripke_witness_t *witness;
};

__global__ void __launch_bounds__(128) finish_frames_kernel(FramesFinishParams p) {
    const uint32_t rec = blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5);
    const uint32_t lane = threadIdx.x & 31u;
    if (rec >= p.n_records) return;
    const Accum a = p.accum[rec];
    uint64_t wf = KRIPKE_NO_WITNESS;
    uint32_t wv = 0, ww = 0;
    if (a.best != ~0ull) {
        const uint32_t fa = p.pairs ? p.pairs[2 * rec] : rec, fb = p.pairs ? p.pairs[2 * rec + 1] : rec;
        const uint8_t *ca = p.code + p.offsets[fa], *cb = p.code + p.offsets[fb];
        const uint32_t la = p.offsets[fa + 1] - p.offsets[fa], lb = p.offsets[fb + 1] - p.offsets[fb];
        const uint32_t full = (1u << p.n) - 1u;
        const uint64_t nval = 1ull << (p.k * p.n);
        uint32_t succ[KRIPKE_LIST_MAX_WORLDS];
        for (uint32_t w = 0; w < p.n; ++w) succ[w] = p.succ[a.best * p.n + w];
        for (uint64_t base = 0; base < nval; base += 32) {
            const uint64_t v = base + lane;
            uint32_t fail = 0;
            if (v < nval) {
                uint32_t val[KRIPKE_MAX_VARS];
                for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) val[i] = (uint32_t)(v >> (i * p.n)) & full;
                const uint32_t t = eval_postfix_scalar(ca, la, p.n, succ, val, full);
                fail = p.pairs ? (t ^ eval_postfix_scalar(cb, lb, p.n, succ, val, full)) : (full & ~t);
            }
            const uint32_t bal = __ballot_sync(0xFFFFFFFFu, fail != 0u);
            if (bal) {
                const int src = __ffs(bal) - 1;
                wf = p.index_base + a.best;
                wv = (uint32_t)(base + src);
                ww = __ffs(__shfl_sync(0xFFFFFFFFu, fail, src)) - 1;
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

}  // namespace

// Valuations per pass: 4 for n <= 9 (registers and spill columns still leave several resident
// blocks), else 2, else 1 (variable-free programs have a single valuation).
int launch_frames(const FramesJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches) {
    const uint32_t bits = job.k * job.n;
    const int vb = (bits >= 2 && job.n <= 9) ? 4 : (bits >= 1 ? 2 : 1);
    switch (job.n) {
#define FR_CASE(N) \
    case N: return vb == 4 ? launch_frames_##N##_v4(job, plan, stream, launches) \
                 : vb == 2 ? launch_frames_##N##_v2(job, plan, stream, launches) \
                           : launch_frames_##N##_v1(job, plan, stream, launches);
        FR_CASE(1) FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7) FR_CASE(8)
        FR_CASE(9) FR_CASE(10) FR_CASE(11) FR_CASE(12) FR_CASE(13) FR_CASE(14) FR_CASE(15) FR_CASE(16)
#undef FR_CASE
    }
    return 801;   // cudaErrorNotSupported
}

int launch_frames_scalar(const FramesJob &job, const uint32_t *records, uint32_t n_list, void *stream,
                         uint32_t *launches) {
    if (n_list == 0 || job.n_frames == 0) return 0;
    FramesScalarParams p;
    p.succ = job.succ; p.n_frames = job.n_frames; p.n = job.n; p.k = job.k;
    p.code = job.code; p.offsets = job.offsets; p.pairs = job.pairs;
    p.records = records; p.n_list = n_list; p.accum = job.accum;
    const uint64_t blocks = std::min<uint64_t>((job.n_frames + 127) / 128, 148ull * 16);
    scan_frames_scalar_kernel<<<(uint32_t)blocks, 128, 0, (cudaStream_t)stream>>>(p);
    if (launches) ++*launches;
    return (int)cudaGetLastError();
}

int launch_frames_finish(const FramesJob &job, bool accumulate, kripke_count_t *counts_out,
                         kripke_witness_t *witness_out, void *stream) {
    if (job.n_records == 0) return 0;
    FramesFinishParams p;
    p.succ = job.succ; p.n = job.n; p.k = job.k;
    p.code = job.code; p.offsets = job.offsets; p.pairs = job.pairs;
    p.n_records = job.n_records; p.accum = job.accum;
    p.index_base = job.index_base; p.accumulate = accumulate;
    p.counts = counts_out; p.witness = witness_out;
    finish_frames_kernel<<<(job.n_records + 3) / 4, 128, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

}  // namespace kripke
