// scan_frames.cu - frame-list mode: the fused evaluator over EXPLICIT frames of up to 16 worlds
// (survivors of the exhaustive prefix are "challenged on paths, reverse paths,
// looped paths, and forked paths of six to ten worlds" / "39 ... templates at each size from six
// through sixteen"; Table 2: synthesized relations, 8,995,007 of them).
//
// Here frames are data (n successor masks each, 2n bytes), so the layout is the transpose of the
// census kernel's: a 32-bit word carries one truth bit for 32 consecutive FRAMES of the list, a
// truth set is N words, and the valuation is block-uniform (atoms are all-0 / all-1 words).  Lemma
// 1 on 32 frames at once is the same N*N three-input logic instructions as in scan_sliced.cuh,
//     box: R[w] = AND_u ( T[u] | ~E[w][u] )        dia: R[w] = OR_u ( T[u] & E[w][u] )
// with E[w][u] = the word of edge bits w->u of the thread's 32 frames.  A block reads its tile of
// TPB*32 frames from HBM once (coalesced 16-bit masks), transposes it on chip with warp ballots
// into a shared-memory table E[w*N+u][thread], and then runs every program of its chunk and every
// valuation against that table: HBM traffic is 2n bytes per frame per program chunk, the inner
// loop reads one shared-memory word per logic instruction.
//
// Programs are the same lowered micro-ops as the census kernel's (ucode.h, lowered without derived
// leaves).  The top of the register stack lives in registers A[N]; deeper slots are spilled to a
// per-thread shared-memory column when a load pushes (the lowering is stack-disciplined: a load
// into slot d happens exactly when slot d-1 is the top).
#include <cuda_runtime.h>

#include <algorithm>

#include "frames.cuh"
#include "internal.h"

namespace kripke {

namespace {

constexpr int FR_TPB = 128;                     // threads per block = groups of 32 frames per tile
constexpr int FR_SPILL = UC_DMAX - 1;           // stack slots below the top

struct FramesParams {
    const uint16_t *succ;          // n_frames * N masks
    uint64_t n_frames;
    uint32_t k;
    const uint16_t *ucode;
    const uint32_t *slot_record;
    uint32_t n_slots, stride;
    uint32_t chunk, n_chunks;      // slots per work item
    uint32_t n_tiles;              // tiles of FR_TPB * 32 frames
    Accum *accum;
};

template <int F> __device__ __forceinline__ uint32_t bfn(uint32_t a, uint32_t b) {
    return (F == BF_AND) ? (a & b) : (F == BF_OR) ? (a | b) : (F == BF_ANDN) ? (a & ~b) : (~a & b);
}
__device__ __forceinline__ uint32_t bfn_rt(uint32_t f, uint32_t a, uint32_t b) {
    return (f == BF_AND) ? (a & b) : (f == BF_OR) ? (a | b) : (f == BF_ANDN) ? (a & ~b) : (~a & b);
}

template <int N>
struct FramesThread {
    uint32_t A[N];                 // top of the stack
    const uint32_t *E;             // this thread's column of the edge table: E[(w*N+u)*FR_TPB]
    uint32_t *S;                   // this thread's spill column: S[(d*N+w)*FR_TPB]

    __device__ __forceinline__ void push(uint32_t d) {          // a load into slot d > 0 pushes
        if (d == 0) return;
#pragma unroll
        for (int w = 0; w < N; ++w) S[((d - 1) * N + w) * FR_TPB] = A[w];
    }
    __device__ __forceinline__ void box() {
        uint32_t r[N];
#pragma unroll
        for (int w = 0; w < N; ++w) {
            uint32_t acc = 0xFFFFFFFFu;
#pragma unroll
            for (int u = 0; u < N; ++u) acc &= (A[u] | ~E[(w * N + u) * FR_TPB]);
            r[w] = acc;
        }
#pragma unroll
        for (int w = 0; w < N; ++w) A[w] = r[w];
    }
    __device__ __forceinline__ void dia() {
        uint32_t r[N];
#pragma unroll
        for (int w = 0; w < N; ++w) {
            uint32_t acc = 0u;
#pragma unroll
            for (int u = 0; u < N; ++u) acc |= (A[u] & E[(w * N + u) * FR_TPB]);
            r[w] = acc;
        }
#pragma unroll
        for (int w = 0; w < N; ++w) A[w] = r[w];
    }

    // One lowered program on the thread's 32 frames under valuation v; returns the word of frames
    // that refute the formula / distinguish the pair.
    __device__ __forceinline__ uint32_t run(const uint16_t *__restrict__ uc, uint32_t v) {
        uint32_t pc = 0, nxt = uc[0], op;
        for (;;) {
            op = nxt & 0xFFu;
            if (op >= (uint32_t)UC_FIN_ALL && op <= (uint32_t)UC_FIN_XNOR) break;
            nxt = uc[++pc];
            if (op < (uint32_t)UC_BOOLV) {                       // LOADV + i*4 + d
                const uint32_t i = op >> 2;
                push(op & 3u);
#pragma unroll
                for (int w = 0; w < N; ++w) A[w] = 0u - ((v >> (i * N + w)) & 1u);
            } else if (op < (uint32_t)UC_LOADL) {                // BOOLV + (f*4 + i)*4 + d
                const uint32_t x = op - UC_BOOLV, i = (x >> 2) & 3u, f = x >> 4;
#pragma unroll
                for (int w = 0; w < N; ++w) A[w] = bfn_rt(f, A[w], 0u - ((v >> (i * N + w)) & 1u));
            } else if (op >= (uint32_t)UC_BOOL && op < (uint32_t)UC_BOX) {   // BOOL + f*4 + d
                const uint32_t x = op - UC_BOOL, d = x & 3u, f = x >> 2;
#pragma unroll
                for (int w = 0; w < N; ++w) A[w] = bfn_rt(f, S[(d * N + w) * FR_TPB], A[w]);
            } else if (op >= (uint32_t)UC_BOX && op < (uint32_t)UC_DIA) {
                box();
            } else if (op >= (uint32_t)UC_DIA && op < (uint32_t)UC_FIN_ALL) {
                dia();
            } else if (op >= (uint32_t)UC_LOADZ) {               // LOADZ + d
                push(op - UC_LOADZ);
#pragma unroll
                for (int w = 0; w < N; ++w) A[w] = 0u;
            }
            // UC_LOADL / UC_BOOLL are never emitted: the programs are lowered without derived leaves
        }
        const uint32_t kind = op - UC_FIN_ALL;
        const uint32_t pol = ((kind ^ (kind >> 1)) & 1u) ? 0u : 0xFFFFFFFFu;
        uint32_t x = 0u;
        if (kind >= 2u) {
#pragma unroll
            for (int w = 0; w < N; ++w) x |= S[w * FR_TPB] ^ A[w] ^ pol;
        } else {
#pragma unroll
            for (int w = 0; w < N; ++w) x |= A[w] ^ pol;
        }
        return x;
    }
};

template <int N>
__global__ void __launch_bounds__(FR_TPB) scan_frames_kernel(FramesParams p) {
    extern __shared__ __align__(16) unsigned char smem[];
    // [E: N*N x TPB][spill: FR_SPILL*N x TPB][valid: TPB][models u64 x chunk][frames u32][best u32][ucode]
    uint32_t *s_E = reinterpret_cast<uint32_t *>(smem);
    uint32_t *s_S = s_E + N * N * FR_TPB;
    uint32_t *s_valid = s_S + FR_SPILL * N * FR_TPB;
    unsigned long long *s_models = reinterpret_cast<unsigned long long *>(s_valid + FR_TPB);
    uint32_t *s_frames = reinterpret_cast<uint32_t *>(s_models + p.chunk);
    uint32_t *s_best = s_frames + p.chunk;
    uint16_t *s_ucode = reinterpret_cast<uint16_t *>(s_best + p.chunk);

    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t n_items = p.n_tiles * p.n_chunks;
    const uint32_t nval = 1u << (p.k * N);
    FramesThread<N> T;
    T.E = s_E + threadIdx.x;
    T.S = s_S + threadIdx.x;

    for (uint32_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        const uint32_t chunk_id = item % p.n_chunks, tile = item / p.n_chunks;
        const uint32_t slot0 = chunk_id * p.chunk;
        const uint32_t nslots = min(p.chunk, p.n_slots - slot0);
        const uint64_t frame0 = (uint64_t)tile * (FR_TPB * 32);

        __syncthreads();
        for (uint32_t i = threadIdx.x; i < nslots; i += FR_TPB) {
            s_models[i] = 0ull; s_frames[i] = 0u; s_best[i] = 0xFFFFFFFFu;
        }
        {
            const uint32_t words = nslots * (p.stride / 2);
            const uint32_t *src = reinterpret_cast<const uint32_t *>(p.ucode + (size_t)slot0 * p.stride);
            uint32_t *dst = reinterpret_cast<uint32_t *>(s_ucode);
            for (uint32_t i = threadIdx.x; i < words; i += FR_TPB) dst[i] = src[i];
        }
        // the tile's frames -> bit-sliced edge table: warp `warp` transposes the groups of its own
        // 32 threads, one group (32 frames, one per lane) at a time
        for (uint32_t gi = 0; gi < 32; ++gi) {
            const uint32_t t = warp * 32 + gi;
            const uint64_t j = frame0 + (uint64_t)t * 32 + lane;
            const bool valid = j < p.n_frames;
            uint32_t m[N];
#pragma unroll
            for (int w = 0; w < N; ++w) m[w] = valid ? (uint32_t)__ldg(p.succ + j * N + w) : 0u;
            const uint32_t vm = __ballot_sync(0xFFFFFFFFu, valid);
            if (lane == 0) s_valid[t] = vm;
#pragma unroll
            for (int w = 0; w < N; ++w)
#pragma unroll
                for (int u = 0; u < N; ++u) {
                    const uint32_t word = __ballot_sync(0xFFFFFFFFu, (m[w] >> u) & 1u);
                    if (lane == (uint32_t)((w * N + u) & 31)) s_E[(w * N + u) * FR_TPB + t] = word;
                }
        }
        __syncthreads();

        const uint32_t vmask = s_valid[threadIdx.x];
        const bool warp_live = __ballot_sync(0xFFFFFFFFu, vmask != 0u) != 0u;   // else: whole warp past the end
        for (uint32_t s = 0; warp_live && s < nslots; ++s) {
            const uint16_t *uc = s_ucode + s * p.stride;
            uint32_t cnt = 0, any = 0;
            for (uint32_t v = 0; v < nval; ++v) {
                const uint32_t r = T.run(uc, v) & vmask;
                cnt += __popc(r);
                any |= r;
            }
            const uint32_t bal = __ballot_sync(0xFFFFFFFFu, any != 0u);
            if (bal) {
                const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, cnt);
                const uint32_t ftot = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)__popc(any));
                const uint32_t first = __shfl_sync(0xFFFFFFFFu, any, __ffs(bal) - 1);
                if (lane == 0) {
                    atomicAdd(&s_models[s], (unsigned long long)tot);
                    atomicAdd(&s_frames[s], ftot);
                    atomicMin(&s_best[s], (warp * 32 + (uint32_t)(__ffs(bal) - 1)) * 32 + (uint32_t)(__ffs(first) - 1));
                }
            }
        }
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < nslots; i += FR_TPB) {
            if (s_best[i] != 0xFFFFFFFFu) {
                Accum *a = p.accum + p.slot_record[slot0 + i];
                atomicAdd(&a->models, s_models[i]);
                atomicAdd(&a->frames, (unsigned long long)s_frames[i]);
                atomicMin(&a->best, frame0 + s_best[i]);
            }
        }
    }
}

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

template <int N>
int launch_frames_n(const FramesJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches) {
    static int sm_count = 0;
    static size_t smem_max = 0;
    auto kern = scan_frames_kernel<N>;
    const size_t fixed = ((size_t)N * N + (size_t)FR_SPILL * N + 1) * FR_TPB * sizeof(uint32_t);
    const size_t per_slot = 16 + 2 * (size_t)plan.stride;
    if (!sm_count) {
        int dev = 0, optin = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
        if (e != cudaSuccess) return (int)e;
        smem_max = std::min<size_t>((size_t)optin, fixed + 32 * 1024 + 16);
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
        if (e != cudaSuccess) return (int)e;
    }
    FramesParams p;
    p.succ = job.succ; p.n_frames = job.n_frames; p.k = job.k;
    p.ucode = plan.ucode; p.slot_record = plan.slot_record;
    p.n_slots = plan.n_slots; p.stride = plan.stride;
    p.accum = job.accum;
    if (p.n_frames == 0 || p.n_slots == 0) return 0;
    const uint64_t tiles = (p.n_frames + FR_TPB * 32 - 1) / (FR_TPB * 32);
    if (tiles > 0x7FFFFFFFull / 4096) return 801;                  // cudaErrorNotSupported
    p.n_tiles = (uint32_t)tiles;
    const uint32_t chunk_cap = (uint32_t)std::max<size_t>(1, std::min<size_t>(2048, (smem_max - fixed - 16) / per_slot));
    // enough work items to fill the grid (two resident blocks per SM at most), each as large as allowed
    const uint64_t want_items = (uint64_t)sm_count * 4;
    uint64_t want_chunks = (want_items + tiles - 1) / tiles;
    uint32_t chunk = (uint32_t)std::max<uint64_t>(1, (p.n_slots + want_chunks - 1) / want_chunks);
    chunk = std::min(std::min(chunk, chunk_cap), p.n_slots);
    p.chunk = chunk;
    p.n_chunks = (p.n_slots + chunk - 1) / chunk;
    const uint64_t items = tiles * p.n_chunks;
    const uint32_t grid = (uint32_t)std::min<uint64_t>(items, (uint64_t)sm_count * 2);
    const size_t smem = fixed + (size_t)chunk * per_slot + 16;
    kern<<<grid, FR_TPB, smem, (cudaStream_t)stream>>>(p);
    if (launches) ++*launches;
    return (int)cudaGetLastError();
}

}  // namespace

int launch_frames(const FramesJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches) {
    switch (job.n) {
#define FR_CASE(N) case N: return launch_frames_n<N>(job, plan, stream, launches);
        FR_CASE(1) FR_CASE(2) FR_CASE(3) FR_CASE(4) FR_CASE(5) FR_CASE(6) FR_CASE(7) FR_CASE(8)
        FR_CASE(9) FR_CASE(10) FR_CASE(11) FR_CASE(12) FR_CASE(13) FR_CASE(14) FR_CASE(15) FR_CASE(16)
#undef FR_CASE
    }
    return 801;
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
