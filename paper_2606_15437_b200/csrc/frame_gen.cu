// frame_gen.cu - in-library generators of explicit frame lists ("paths,
// reverse paths, looped paths, and forked paths" / "path, reverse-path, reflexive-path, fork, cycle, star,
// sparse, and dense templates"; "stratified Erdos-Renyi sampling, edge-flip mutation of canonical
// seeds, ... dead-end insertion, back-edge injection").  One thread writes one frame as n successor masks in the
// format of kripke_eval_frames, so a stress list never exists on the host.  Random choices come from a
// counter-based generator (SplitMix64 finaliser of seed, generator, size, frame position, draw index), which
// workloads/frames.py restates in numpy for the oracle side: the lists are inputs, not part of the method.
#include <cuda_runtime.h>

#include "internal.h"

namespace kripke {

namespace {

__host__ __device__ inline unsigned long long gen_mix(unsigned long long x) {
    x += 0x9E3779B97F4A7C15ull;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ull;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

struct Draw {
    unsigned long long key, j;
    __device__ Draw(unsigned long long seed, uint32_t gen, uint32_t n, unsigned long long j_)
        : key(gen_mix(seed ^ ((unsigned long long)gen << 56) ^ ((unsigned long long)n << 48))), j(j_) {}
    __device__ unsigned long long operator()(uint32_t t) const {
        return gen_mix(key + j * 0xD6E8FEB86659FD93ull + (unsigned long long)t * 0x2545F4914F6CDD1Dull);
    }
};

// densities 0.05, 0.1, 0.2, 0.35, 0.5, 0.8 and 0.3 as thresholds on the upper 32 bits of a draw
__constant__ uint32_t kDensity[6] = {214748364u, 429496729u, 858993459u, 1503238553u, 2147483648u, 3435973836u};
constexpr uint32_t kDensity03 = 1288490188u;

__device__ void template_rows(uint32_t kind, uint32_t n, uint32_t *row) {
    for (uint32_t w = 0; w < n; ++w) row[w] = 0;
    const uint32_t full = (n >= 32) ? 0xFFFFFFFFu : ((1u << n) - 1u);
    switch (kind) {
    case KRIPKE_TPL_PATH: case KRIPKE_TPL_REFLEXIVE_PATH: case KRIPKE_TPL_CYCLE: case KRIPKE_TPL_PATH_LOOP_END:
        for (uint32_t w = 0; w + 1 < n; ++w) row[w] = 1u << (w + 1);
        if (kind == KRIPKE_TPL_REFLEXIVE_PATH) for (uint32_t w = 0; w < n; ++w) row[w] |= 1u << w;
        if (kind == KRIPKE_TPL_CYCLE) row[n - 1] |= 1u;
        if (kind == KRIPKE_TPL_PATH_LOOP_END) row[n - 1] |= 1u << (n - 1);
        break;
    case KRIPKE_TPL_REVERSE_PATH:
        for (uint32_t w = 1; w < n; ++w) row[w] = 1u << (w - 1);
        break;
    case KRIPKE_TPL_FORK:
        if (n < 3) { for (uint32_t w = 0; w + 1 < n; ++w) row[w] = 1u << (w + 1); break; }
        for (uint32_t w = 0; w + 3 < n; ++w) row[w] = 1u << (w + 1);
        row[n - 3] = (1u << (n - 2)) | (1u << (n - 1));
        break;
    case KRIPKE_TPL_STAR: row[0] = full & ~1u; break;
    case KRIPKE_TPL_REVERSE_STAR: for (uint32_t w = 1; w < n; ++w) row[w] = 1u; break;
    case KRIPKE_TPL_COMPLETE: for (uint32_t w = 0; w < n; ++w) row[w] = full; break;
    default: break;                                                   // KRIPKE_TPL_EMPTY
    }
}

__device__ void generate_one(uint32_t gen, uint32_t n, unsigned long long j, unsigned long long seed, uint32_t *row) {
    const Draw d(seed, gen, n, j);
    switch (gen) {
    case KRIPKE_GEN_TEMPLATES:
        template_rows((uint32_t)(j % KRIPKE_TPL_COUNT), n, row);
        break;
    case KRIPKE_GEN_ERDOS_RENYI: case KRIPKE_GEN_DEAD_END: {
        const uint32_t thr = gen == KRIPKE_GEN_ERDOS_RENYI ? kDensity[j % 6] : kDensity03;
        for (uint32_t w = 0; w < n; ++w) {
            uint32_t r = 0;
            for (uint32_t u = 0; u < n; ++u) r |= (uint32_t)((uint32_t)(d(w * n + u) >> 32) < thr) << u;
            row[w] = r;
        }
        if (gen == KRIPKE_GEN_DEAD_END) row[d(1000) % n] = 0;
        break;
    }
    case KRIPKE_GEN_EDGE_FLIP: {
        template_rows((uint32_t)(j % KRIPKE_TPL_COUNT), n, row);
        const uint32_t flips = 1 + (uint32_t)(d(100) % 4);
        for (uint32_t t = 0; t < flips; ++t) {
            const uint32_t pos = (uint32_t)(d(t) % (n * n));
            row[pos / n] ^= 1u << (pos % n);
        }
        break;
    }
    default: {                                                        // KRIPKE_GEN_BACK_EDGE
        template_rows(KRIPKE_TPL_PATH, n, row);
        for (uint32_t t = 0; t < 2; ++t) {
            const uint32_t w = (uint32_t)(d(2 * t) % n);
            const uint32_t u = (uint32_t)(d(2 * t + 1) % (w + 1));
            row[w] |= 1u << u;
        }
    }
    }
}

__global__ void frames_generate_kernel(uint32_t gen, uint32_t n, unsigned long long n_frames, unsigned long long seed,
                                       uint16_t *succ) {
    const unsigned long long j = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n_frames) return;
    uint32_t row[KRIPKE_LIST_MAX_WORLDS];
    if (gen != KRIPKE_GEN_STRESS) {
        generate_one(gen, n, j, seed, row);
    } else {
        // the mixed list: the templates, then the four generators in equal shares (workloads/frames.py stress_list_cb)
        const unsigned long long nt = n_frames < KRIPKE_TPL_COUNT ? n_frames : KRIPKE_TPL_COUNT;
        if (j < nt) {
            generate_one(KRIPKE_GEN_TEMPLATES, n, j, seed, row);
        } else {
            const unsigned long long rest = n_frames - nt;
            unsigned long long r = j - nt;
            uint32_t part = 0;
            for (; part < 4; ++part) {
                const unsigned long long q = rest / 4 + (part < rest % 4 ? 1 : 0);
                if (r < q) break;
                r -= q;
            }
            generate_one(KRIPKE_GEN_ERDOS_RENYI + part, n, r, seed, row);
        }
    }
    for (uint32_t w = 0; w < n; ++w) succ[j * n + w] = (uint16_t)row[w];
}

}  // namespace

int launch_frames_generate(uint32_t gen, uint32_t n, uint64_t n_frames, uint64_t seed, uint16_t *succ_out, void *stream) {
    if (n_frames == 0) return 0;
    const uint64_t blocks = (n_frames + 255) / 256;
    frames_generate_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(gen, n, n_frames, seed, succ_out);
    return (int)cudaGetLastError();
}

}  // namespace kripke
