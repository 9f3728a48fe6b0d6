// scan_frames.cuh - frame-list mode, bit-sliced kernel: the fused evaluator over EXPLICIT frames of
// up to 16 worlds (survivors of the exhaustive prefix are "challenged on paths,
// reverse paths, looped paths, and forked paths of six to ten worlds" / "39 ... templates at each
// size from six through sixteen"; Table 2: 8,995,007 synthesized relations).
//
// Layout.  Frames are data here (n successor masks each, 2n bytes), so the layout is the transpose
// of the census kernel's: a 32-bit word carries one truth bit for 32 consecutive FRAMES of the
// list, a truth set is N words, and the valuation is warp-uniform (atoms are all-0 / all-1 words).
// Lemma 1 on 32 frames at once is the same N*N three-input logic instructions as in
// scan_sliced.cuh,
//     box: R[w] = AND_u ( T[u] | ~E[w][u] )        dia: R[w] = OR_u ( T[u] & E[w][u] )
// with E[w][u] = the word of edge bits w->u of the lane's 32 frames.
//
// Work decomposition.  A work item is (tile of 32 x 32 = 1,024 consecutive frames) x (chunk of
// programs).  The block reads the tile's masks from HBM once (2n bytes per frame), transposes them
// on chip with warp ballots into a shared-memory edge table E[w*N+u][lane] (N*N*128 bytes: 32 KB
// at n = 16), and its four warps then take the chunk's programs from a shared work counter, every
// warp against the same table: lane = group of 32 frames, so the table reads are conflict-free and the table is
// shared by all warps (small footprint -> several resident blocks per SM).  One shared-memory word
// feeds VB logic instructions: a pass evaluates VB consecutive valuations (VB = 4 or 2 when the
// programs have variables), whose atoms differ only in compile-time bits.
//
// Programs are the census kernel's lowered micro-ops (ucode.h), lowered without derived leaves.
// The top of the register stack lives in registers A[VB][N]; deeper slots are spilled to a
// per-thread shared-memory column when a load pushes (the lowering is stack-disciplined: a load
// into slot d happens exactly when slot d-1 is the top).  Reduction: per (warp, program, tile)
// popcounts -> __reduce_add_sync -> one global atomic triple, skipped when nothing in the tile
// refutes.
#pragma once
#include <cuda_runtime.h>

#include <algorithm>

#include "internal.h"

namespace kripke {

constexpr int FR_TPB = 128;                     // four warps per block
constexpr int FR_WARPS = FR_TPB / 32;
constexpr int FR_SPILL = UC_DMAX - 1;           // stack slots below the top

struct FramesParams {
    const uint16_t *succ;          // n_frames * N masks
    uint64_t n_frames;
    uint32_t k;
    const uint16_t *ucode;
    const uint32_t *slot_record;
    uint32_t n_slots, stride;
    uint32_t chunk, n_chunks;      // slots per work item
    uint32_t n_tiles;              // tiles of 1,024 frames
    uint32_t spill_slots;          // stack slots kept below the top (max need - 1, <= FR_SPILL)
    Accum *accum;
};

template <int N, int VB>
struct FramesThread {
    static constexpr int LOGVB = VB == 4 ? 2 : VB == 2 ? 1 : 0;
    uint32_t A[VB][N];             // top of the stack, one truth set per valuation of the pass
    const uint32_t *E;             // this lane's column of the edge table: E[(w*N+u)*32]
    uint32_t *S;                   // this thread's spill column: S[((d*N+w)*VB+j)*FR_TPB]

    // word of "p_i holds at world w" under valuation v0 + j (v0 a multiple of VB)
    __device__ __forceinline__ uint32_t atom(uint32_t v0, uint32_t i, int w, int j) const {
        const uint32_t pos = i * N + w;
        const uint32_t bit = pos < (uint32_t)LOGVB ? ((uint32_t)j >> pos) : (v0 >> pos);
        return 0u - (bit & 1u);
    }
    __device__ __forceinline__ void push(uint32_t d) {          // a load into slot d > 0 pushes
        if (d == 0) return;
#pragma unroll
        for (int w = 0; w < N; ++w)
#pragma unroll
            for (int j = 0; j < VB; ++j) S[(((d - 1) * N + w) * VB + j) * FR_TPB] = A[j][w];
    }
    template <int F> static __device__ __forceinline__ uint32_t bf(uint32_t a, uint32_t b) {
        return (F == BF_AND) ? (a & b) : (F == BF_OR) ? (a | b) : (F == BF_ANDN) ? (a & ~b) : (~a & b);
    }
    template <int F> __device__ __forceinline__ void bool_atom(uint32_t v0, uint32_t i) {
#pragma unroll
        for (int w = 0; w < N; ++w)
#pragma unroll
            for (int j = 0; j < VB; ++j) A[j][w] = bf<F>(A[j][w], atom(v0, i, w, j));
    }
    template <int F> __device__ __forceinline__ void bool_slot(uint32_t d) {
#pragma unroll
        for (int w = 0; w < N; ++w)
#pragma unroll
            for (int j = 0; j < VB; ++j) A[j][w] = bf<F>(S[((d * N + w) * VB + j) * FR_TPB], A[j][w]);
    }
    template <bool BOX> __device__ __forceinline__ void modal() {
        uint32_t r[VB][N];
#pragma unroll
        for (int w = 0; w < N; ++w) {
#pragma unroll
            for (int j = 0; j < VB; ++j) r[j][w] = BOX ? 0xFFFFFFFFu : 0u;
#pragma unroll
            for (int u = 0; u < N; ++u) {
                const uint32_t e = E[(w * N + u) * 32];
#pragma unroll
                for (int j = 0; j < VB; ++j) {
                    if (BOX) r[j][w] &= (A[j][u] | ~e);
                    else r[j][w] |= (A[j][u] & e);
                }
            }
        }
#pragma unroll
        for (int j = 0; j < VB; ++j)
#pragma unroll
            for (int w = 0; w < N; ++w) A[j][w] = r[j][w];
    }

    // One lowered program on the lane's 32 frames under valuations v0 .. v0+VB-1; x[j] = the word
    // of frames that refute the formula / distinguish the pair under valuation v0 + j.
    __device__ __forceinline__ void run(const uint16_t *__restrict__ uc, uint32_t v0, uint32_t (&x)[VB]) {
        uint32_t pc = 0, nxt = uc[0], op;
        for (;;) {
            op = nxt & 0xFFu;
            if (op >= (uint32_t)UC_FIN_ALL && op <= (uint32_t)UC_FIN_XNOR) break;
            nxt = uc[++pc];
            if (op < (uint32_t)UC_BOOLV) {                       // LOADV + i*4 + d
                const uint32_t i = op >> 2;
                push(op & 3u);
#pragma unroll
                for (int w = 0; w < N; ++w)
#pragma unroll
                    for (int j = 0; j < VB; ++j) A[j][w] = atom(v0, i, w, j);
            } else if (op < (uint32_t)UC_LOADL) {                // BOOLV + (f*4 + i)*4 + d
                const uint32_t y = op - UC_BOOLV, i = (y >> 2) & 3u, f = y >> 4;
                switch (f) {
                case BF_AND: bool_atom<BF_AND>(v0, i); break;
                case BF_OR: bool_atom<BF_OR>(v0, i); break;
                case BF_ANDN: bool_atom<BF_ANDN>(v0, i); break;
                default: bool_atom<BF_NAND>(v0, i); break;
                }
            } else if (op >= (uint32_t)UC_BOOL && op < (uint32_t)UC_BOX) {   // BOOL + f*4 + d
                const uint32_t y = op - UC_BOOL, d = y & 3u, f = y >> 2;
                switch (f) {
                case BF_AND: bool_slot<BF_AND>(d); break;
                case BF_OR: bool_slot<BF_OR>(d); break;
                case BF_ANDN: bool_slot<BF_ANDN>(d); break;
                default: bool_slot<BF_NAND>(d); break;
                }
            } else if (op >= (uint32_t)UC_BOX && op < (uint32_t)UC_DIA) {
                modal<true>();
            } else if (op >= (uint32_t)UC_DIA && op < (uint32_t)UC_FIN_ALL) {
                modal<false>();
            } else if (op >= (uint32_t)UC_LOADZ) {               // LOADZ + d
                push(op - UC_LOADZ);
#pragma unroll
                for (int w = 0; w < N; ++w)
#pragma unroll
                    for (int j = 0; j < VB; ++j) A[j][w] = 0u;
            }
            // UC_LOADL / UC_BOOLL are never emitted: the programs are lowered without derived leaves
        }
        const uint32_t kind = op - UC_FIN_ALL;                   // 0 ALL, 1 ANY, 2 XOR, 3 XNOR
        const uint32_t pol = ((kind ^ (kind >> 1)) & 1u) ? 0u : 0xFFFFFFFFu;
#pragma unroll
        for (int j = 0; j < VB; ++j) x[j] = 0u;
        if (kind >= 2u) {
#pragma unroll
            for (int w = 0; w < N; ++w)
#pragma unroll
                for (int j = 0; j < VB; ++j) x[j] |= S[(w * VB + j) * FR_TPB] ^ A[j][w] ^ pol;
        } else {
#pragma unroll
            for (int w = 0; w < N; ++w)
#pragma unroll
                for (int j = 0; j < VB; ++j) x[j] |= A[j][w] ^ pol;
        }
    }
};

template <int N, int VB>
__global__ void __launch_bounds__(FR_TPB) scan_frames_kernel(FramesParams p) {
    extern __shared__ __align__(16) unsigned char smem[];
    // [E: N*N x 32][valid: 32][next: 4][spill: spill_slots*N*VB x TPB][ucode]
    uint32_t *s_E = reinterpret_cast<uint32_t *>(smem);
    uint32_t *s_valid = s_E + N * N * 32;
    uint32_t *s_next = s_valid + 32;                    // work counter of the item (one word, padded to 4)
    uint32_t *s_S = s_next + 4;
    uint16_t *s_ucode = reinterpret_cast<uint16_t *>(s_S + p.spill_slots * N * VB * FR_TPB);

    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t n_items = p.n_tiles * p.n_chunks;
    const uint32_t nval = 1u << (p.k * N);
    FramesThread<N, VB> T;
    T.E = s_E + lane;
    T.S = s_S + threadIdx.x;

    for (uint32_t item = blockIdx.x; item < n_items; item += gridDim.x) {
        const uint32_t chunk_id = item % p.n_chunks, tile = item / p.n_chunks;
        const uint32_t slot0 = chunk_id * p.chunk;
        const uint32_t nslots = min(p.chunk, p.n_slots - slot0);
        const uint64_t frame0 = (uint64_t)tile * 1024u;

        __syncthreads();                                  // the previous item's table is no longer read
        {
            const uint32_t words = nslots * (p.stride / 2);
            const uint32_t *src = reinterpret_cast<const uint32_t *>(p.ucode + (size_t)slot0 * p.stride);
            uint32_t *dst = reinterpret_cast<uint32_t *>(s_ucode);
            for (uint32_t i = threadIdx.x; i < words; i += FR_TPB) dst[i] = src[i];
        }
        // the tile's frames -> bit-sliced edge table; each warp transposes 8 of the 32 groups
        for (uint32_t t = warp; t < 32; t += FR_WARPS) {
            const uint64_t j = frame0 + (uint64_t)t * 32 + lane;
            const bool valid = j < p.n_frames;
            uint32_t m[N];
#pragma unroll
            for (int w = 0; w < N; ++w) m[w] = valid ? (uint32_t)__ldg(p.succ + j * N + w) : 0u;
            const uint32_t vm = __ballot_sync(0xFFFFFFFFu, valid);
            if (lane == 0) s_valid[t] = vm;
            if (threadIdx.x == 0) *s_next = 0u;
#pragma unroll
            for (int w = 0; w < N; ++w)
#pragma unroll
                for (int u = 0; u < N; ++u) {
                    const uint32_t word = __ballot_sync(0xFFFFFFFFu, (m[w] >> u) & 1u);
                    if (lane == (uint32_t)((w * N + u) & 31)) s_E[(w * N + u) * 32 + t] = word;
                }
        }
        __syncthreads();

        const uint32_t vmask = s_valid[lane];
        // the chunk's programs go to whichever warp is free next (programs differ in length)
        for (;;) {
            uint32_t s = 0;
            if (lane == 0) s = atomicAdd(s_next, 1u);
            s = __shfl_sync(0xFFFFFFFFu, s, 0);
            if (s >= nslots) break;
            const uint16_t *uc = s_ucode + s * p.stride;
            uint32_t cnt = 0, any = 0;
            for (uint32_t v0 = 0; v0 < nval; v0 += VB) {
                uint32_t x[VB];
                T.run(uc, v0, x);
#pragma unroll
                for (int j = 0; j < VB; ++j) {
                    const uint32_t r = x[j] & vmask;
                    cnt += __popc(r);
                    any |= r;
                }
            }
            const uint32_t bal = __ballot_sync(0xFFFFFFFFu, any != 0u);
            if (bal) {
                const uint32_t tot = __reduce_add_sync(0xFFFFFFFFu, cnt);
                const uint32_t ftot = __reduce_add_sync(0xFFFFFFFFu, (uint32_t)__popc(any));
                const uint32_t first = __shfl_sync(0xFFFFFFFFu, any, __ffs(bal) - 1);
                if (lane == 0) {
                    Accum *a = p.accum + p.slot_record[slot0 + s];
                    atomicAdd(&a->models, (unsigned long long)tot);
                    atomicAdd(&a->frames, (unsigned long long)ftot);
                    atomicMin(&a->best, frame0 + (uint64_t)(__ffs(bal) - 1) * 32 + (uint64_t)(__ffs(first) - 1));
                }
            }
        }
    }
}

// Host launcher for one instantiation.
template <int N, int VB>
int launch_frames_inst(const FramesJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches) {
    // queried for the current device on every call (nothing cached per process: multi-device / multi-thread safe)
    int sm_count = 0, blocks_per_sm[FR_SPILL + 1] = {0, 0, 0, 0};
    auto kern = scan_frames_kernel<N, VB>;
    const uint32_t spill_slots = std::min<uint32_t>(FR_SPILL, plan.max_need > 0 ? plan.max_need - 1 : 0);
    const size_t fixed = ((size_t)N * N * 32 + 36 + (size_t)spill_slots * N * VB * FR_TPB) * sizeof(uint32_t);
    const size_t slot_budget = 8 * 1024;
    {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        const size_t most = ((size_t)N * N * 32 + 36 + (size_t)FR_SPILL * N * VB * FR_TPB) * sizeof(uint32_t);
        e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(most + slot_budget));
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&sm_count, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return (int)e;
    }
    {
        int b = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, kern, FR_TPB, fixed + slot_budget);
        if (e != cudaSuccess) return (int)e;
        blocks_per_sm[spill_slots] = b > 0 ? b : 1;
    }
    FramesParams p;
    p.succ = job.succ; p.n_frames = job.n_frames; p.k = job.k;
    p.ucode = plan.ucode; p.slot_record = plan.slot_record;
    p.n_slots = plan.n_slots; p.stride = plan.stride;
    p.accum = job.accum;
    p.spill_slots = spill_slots;
    if (p.n_frames == 0 || p.n_slots == 0) return 0;
    const uint64_t tiles = (p.n_frames + 1023) / 1024;
    p.n_tiles = (uint32_t)tiles;
    const uint32_t chunk_cap = (uint32_t)std::max<size_t>(FR_WARPS, slot_budget / (2 * (size_t)plan.stride));
    // enough work items to fill the grid a few times over, each chunk a multiple of the warp count
    const uint64_t grid_full = (uint64_t)sm_count * blocks_per_sm[spill_slots];
    const uint64_t want_chunks = std::max<uint64_t>(1, (grid_full * 4 + tiles - 1) / tiles);
    uint64_t chunk = (p.n_slots + want_chunks - 1) / want_chunks;
    chunk = (chunk + FR_WARPS - 1) / FR_WARPS * FR_WARPS;
    chunk = std::min<uint64_t>(std::min<uint64_t>(chunk, chunk_cap / FR_WARPS * FR_WARPS), std::max<uint32_t>(p.n_slots, 1));
    p.chunk = (uint32_t)std::max<uint64_t>(1, chunk);
    p.n_chunks = (p.n_slots + p.chunk - 1) / p.chunk;
    const uint64_t items = tiles * p.n_chunks;
    if (items > 0x7FFFFFFFull) return 801;                         // cudaErrorNotSupported
    const uint32_t grid = (uint32_t)std::min<uint64_t>(items, grid_full);
    const size_t smem = fixed + (size_t)p.chunk * 2 * plan.stride;
    kern<<<grid, FR_TPB, smem, (cudaStream_t)stream>>>(p);
    if (launches) ++*launches;
    return (int)cudaGetLastError();
}

}  // namespace kripke
