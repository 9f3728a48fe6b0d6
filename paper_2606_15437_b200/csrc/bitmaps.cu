// bitmaps.cu - correspondence recovery (Table 9 at PAPER.md:366-376; SURVEY.md 8f
// N3): per-formula frame-validity bitmaps over a class range, bitmaps of first-order frame
// conditions over the same range, and the matching of the former against a library of the latter.
// One bit per class frame, bit (j % 32) of word (j / 32) = frame frame_begin + j; the bits past the
// range in the last word are 0 in both kinds of bitmap, so equal bitmaps compare equal word by word.
#include <cuda_runtime.h>

#include <algorithm>

#include "frames.cuh"
#include "internal.h"

namespace kripke {

namespace {

__device__ __forceinline__ void decode_rows(uint32_t n, uint64_t f, uint32_t *succ) {
    const uint32_t full = (1u << n) - 1u;
    for (uint32_t w = 0; w < n; ++w) succ[w] = (uint32_t)(f >> (w * n)) & full;
}

// Validity: thread = frame; a formula is valid on the frame iff no valuation gives a truth set other
// than W; the valuation loop stops at the first refutation.  blockIdx.y strides over
// the formulas.  One ballot per (warp, formula) is the output word.
struct ValidityParams {
    uint32_t n, k, cls;
    const uint64_t *class_table;
    uint64_t frame_begin, frame_count;
    const uint8_t *code;
    const uint32_t *offsets;
    uint32_t n_formulas;
    uint32_t *bitmap;
    uint64_t words;               // per formula
};

__global__ void __launch_bounds__(128) validity_bitmap_kernel(ValidityParams p) {
    const uint32_t lane = threadIdx.x & 31u;
    const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;        // position in the range
    const bool in_range = j < p.frame_count;
    const uint32_t full = (1u << p.n) - 1u;
    const uint64_t nval = 1ull << (p.k * p.n);
    uint32_t succ[KRIPKE_MAX_WORLDS];
    decode_rows(p.n, class_frame(p.n, p.cls, p.class_table, p.frame_begin + (in_range ? j : 0)), succ);
    for (uint32_t b = blockIdx.y; b < p.n_formulas; b += gridDim.y) {
        const uint8_t *c = p.code + p.offsets[b];
        const uint32_t len = p.offsets[b + 1] - p.offsets[b];
        bool valid = in_range;
        for (uint64_t v = 0; valid && v < nval; ++v) {
            uint32_t val[KRIPKE_MAX_VARS];
            for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) val[i] = (uint32_t)(v >> (i * p.n)) & full;
            valid = eval_postfix_scalar(c, len, p.n, succ, val, full) == full;
        }
        const uint32_t word = __ballot_sync(0xFFFFFFFFu, valid);
        if (lane == 0 && (j >> 5) < p.words) p.bitmap[(uint64_t)b * p.words + (j >> 5)] = word;
    }
}

// First-order frame conditions on successor masks (the correspondents of Table 9).
__device__ bool frame_condition(uint32_t n, const uint32_t *succ, uint32_t cond) {
    switch (cond) {
    case KRIPKE_COND_REFLEXIVE:                    // every w sees itself
        for (uint32_t w = 0; w < n; ++w) if (!((succ[w] >> w) & 1u)) return false;
        return true;
    case KRIPKE_COND_TRANSITIVE:                   // u in succ[w] => succ[u] subset of succ[w]
        for (uint32_t w = 0; w < n; ++w)
            for (uint32_t u = 0; u < n; ++u)
                if (((succ[w] >> u) & 1u) && (succ[u] & ~succ[w])) return false;
        return true;
    case KRIPKE_COND_SYMMETRIC:
        for (uint32_t w = 0; w < n; ++w)
            for (uint32_t u = w + 1; u < n; ++u)
                if (((succ[w] >> u) & 1u) != ((succ[u] >> w) & 1u)) return false;
        return true;
    case KRIPKE_COND_SERIAL:                       // no dead end
        for (uint32_t w = 0; w < n; ++w) if (succ[w] == 0u) return false;
        return true;
    case KRIPKE_COND_EUCLIDEAN:                    // u in succ[w] => succ[w] subset of succ[u]
        for (uint32_t w = 0; w < n; ++w)
            for (uint32_t u = 0; u < n; ++u)
                if (((succ[w] >> u) & 1u) && (succ[w] & ~succ[u])) return false;
        return true;
    case KRIPKE_COND_PARTIALLY_FUNCTIONAL:         // at most one successor
        for (uint32_t w = 0; w < n; ++w) if (__popc(succ[w]) > 1) return false;
        return true;
    case KRIPKE_COND_DENSE: {                      // succ[w] subset of succ(succ[w])
        for (uint32_t w = 0; w < n; ++w) {
            uint32_t two = 0;
            for (uint32_t u = 0; u < n; ++u) if ((succ[w] >> u) & 1u) two |= succ[u];
            if (succ[w] & ~two) return false;
        }
        return true;
    }
    case KRIPKE_COND_CONFLUENT:                    // two successors of w share a successor
        for (uint32_t w = 0; w < n; ++w)
            for (uint32_t u = 0; u < n; ++u)
                for (uint32_t t = u; t < n; ++t)
                    if (((succ[w] >> u) & 1u) && ((succ[w] >> t) & 1u) && !(succ[u] & succ[t])) return false;
        return true;
    }
    return false;
}

struct ConditionParams {
    uint32_t n, cond, cls;
    const uint64_t *class_table;
    uint64_t frame_begin, frame_count;
    uint32_t *bitmap;
};

__global__ void __launch_bounds__(128) condition_bitmap_kernel(ConditionParams p) {
    const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in_range = j < p.frame_count;
    uint32_t succ[KRIPKE_MAX_WORLDS];
    decode_rows(p.n, class_frame(p.n, p.cls, p.class_table, p.frame_begin + (in_range ? j : 0)), succ);
    const bool holds = in_range && frame_condition(p.n, succ, p.cond);
    const uint32_t word = __ballot_sync(0xFFFFFFFFu, holds);
    if ((threadIdx.x & 31u) == 0 && j < ((p.frame_count + 31) / 32) * 32) p.bitmap[j >> 5] = word;
}

// One warp per record: the index of the first library bitmap equal to the record's, else ~0.
__global__ void __launch_bounds__(128) match_bitmaps_kernel(const uint32_t *bitmaps, uint32_t n_records, uint64_t words,
                                                            const uint32_t *library, uint32_t n_library,
                                                            uint32_t *match_out) {
    const uint32_t rec = blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5);
    const uint32_t lane = threadIdx.x & 31u;
    if (rec >= n_records) return;
    const uint32_t *mine = bitmaps + (uint64_t)rec * words;
    uint32_t found = 0xFFFFFFFFu;
    for (uint32_t l = 0; l < n_library && found == 0xFFFFFFFFu; ++l) {
        const uint32_t *lib = library + (uint64_t)l * words;
        bool same = true;
        for (uint64_t i = lane; i < words && same; i += 32) same = mine[i] == lib[i];
        if (__all_sync(0xFFFFFFFFu, same)) found = l;
    }
    if (lane == 0) match_out[rec] = found;
}

// Failure densities (the atlas matrix): thread = frame, every valuation evaluated with the
// scalar recurrence, count of worlds outside the truth set; blockIdx.y strides the formulas; the store
// counts[b * frames + j] is coalesced over the frames of a warp.  Frames come from the class enumerator
// or, if `succ_list` is set, from an explicit list (n <= 16).
struct DensityParams {
    uint32_t n, k, cls;
    const uint64_t *class_table;
    const uint16_t *succ_list;
    uint64_t frame_begin, frame_count;
    const uint8_t *code;
    const uint32_t *offsets;
    uint32_t n_formulas;              // formulas, or listed records
    const uint32_t *records;          // null = formulas 0..n_formulas-1
    const uint32_t *row_begin, *rows; // not null: listed record i is written to the rows rows[row_begin[i] .. row_begin[i+1])
    uint32_t *counts;
    uint64_t row_stride, col_offset;  // counts[formula * row_stride + col_offset + j]
};

__global__ void __launch_bounds__(128) failure_density_kernel(DensityParams p) {
    const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= p.frame_count) return;
    const uint32_t full = (p.n >= 32 ? 0xFFFFFFFFu : (1u << p.n) - 1u);
    const uint64_t nval = 1ull << (p.k * p.n);
    uint32_t succ[KRIPKE_LIST_MAX_WORLDS];
    if (p.succ_list) {
        for (uint32_t w = 0; w < p.n; ++w) succ[w] = p.succ_list[j * p.n + w];
    } else {
        decode_rows(p.n, class_frame(p.n, p.cls, p.class_table, p.frame_begin + j), succ);
    }
    for (uint32_t li = blockIdx.y; li < p.n_formulas; li += gridDim.y) {
        const uint32_t b = p.records ? p.records[li] : li;
        const uint8_t *c = p.code + p.offsets[b];
        const uint32_t len = p.offsets[b + 1] - p.offsets[b];
        uint32_t cnt = 0;
        for (uint64_t v = 0; v < nval; ++v) {
            uint32_t val[KRIPKE_MAX_VARS];
            for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) val[i] = (uint32_t)(v >> (i * p.n)) & full;
            cnt += __popc(full & ~eval_postfix_scalar(c, len, p.n, succ, val, full));
        }
        if (p.rows) {
            for (uint32_t t = p.row_begin[li]; t < p.row_begin[li + 1]; ++t)
                p.counts[(uint64_t)p.rows[t] * p.row_stride + p.col_offset + j] = cnt;
        } else {
            p.counts[(uint64_t)b * p.row_stride + p.col_offset + j] = cnt;
        }
    }
}

// Frames whose bit is set -> successor masks (input format of the frame-list calls).  Warp-aggregated
// append: the order inside a warp is kept, the order of warps is not.
__global__ void __launch_bounds__(128) frames_from_bitmap_kernel(ConditionParams p, uint16_t *succ_out,
                                                                 unsigned long long capacity,
                                                                 unsigned long long *count_out) {
    const uint64_t j = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t lane = threadIdx.x & 31u;
    const bool set = j < p.frame_count && ((p.bitmap[j >> 5] >> (j & 31u)) & 1u);
    const uint32_t bal = __ballot_sync(0xFFFFFFFFu, set);
    if (bal == 0u) return;
    unsigned long long base = 0;
    if (lane == 0) base = atomicAdd(count_out, (unsigned long long)__popc(bal));
    base = __shfl_sync(0xFFFFFFFFu, base, 0);
    if (!set) return;
    const unsigned long long at = base + (unsigned long long)__popc(bal & ((1u << lane) - 1u));
    if (at >= capacity) return;
    uint32_t succ[KRIPKE_MAX_WORLDS];
    decode_rows(p.n, class_frame(p.n, p.cls, p.class_table, p.frame_begin + j), succ);
    for (uint32_t w = 0; w < p.n; ++w) succ_out[at * p.n + w] = (uint16_t)succ[w];
}

// ---- semantic signatures ("one representative per semantic equivalence class on all frames of
// <= 3 worlds"; "64-bit per-size behaviour fingerprint") ------------------------------------
// One block per formula; its threads stride over every model (frame, valuation) of 1..n_max worlds, evaluate
// the truth set with the scalar recurrence and fold (size, model index, truth set) into two independent
// 64-bit sums.  Addition commutes, so the order of the models - and of the threads - does not matter.  Two
// formulas with equal truth sets on all those models get equal signatures; unequal behaviour collides with
// probability ~2^-128.  The hash only screens: callers that need certainty re-check a class with the pair
// path (kripke_distinguish_pairs over the same sizes), as the paper does ("no equivalence claim
// rests on a matching fingerprint").
__device__ __forceinline__ unsigned long long sig_mix(unsigned long long x) {
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 27; x *= 0x94D049BB133111EBull;
    return x ^ (x >> 31);
}

struct SignatureParams {
    uint32_t k, n_max;
    const uint8_t *code;
    const uint32_t *offsets;
    uint32_t n_formulas;
    unsigned long long *sig;      // 2 per formula
};

__global__ void __launch_bounds__(256) signature_kernel(SignatureParams p) {
    __shared__ unsigned long long s_a[8], s_b[8];
    const uint32_t b = blockIdx.x;
    const uint8_t *c = p.code + p.offsets[b];
    const uint32_t len = p.offsets[b + 1] - p.offsets[b];
    unsigned long long ha = 0, hb = 0;
    for (uint32_t n = 1; n <= p.n_max; ++n) {
        const uint32_t full = (1u << n) - 1u, kn = p.k * n;
        const uint64_t models = 1ull << (n * n + kn);
        for (uint64_t x = threadIdx.x; x < models; x += blockDim.x) {
            const uint64_t f = x >> kn, v = x & ((1ull << kn) - 1ull);
            uint32_t succ[KRIPKE_MAX_WORLDS], val[KRIPKE_MAX_VARS];
            decode_rows(n, f, succ);
            for (uint32_t i = 0; i < KRIPKE_MAX_VARS; ++i) val[i] = (uint32_t)(v >> (i * n)) & full;
            const unsigned long long t = eval_postfix_scalar(c, len, n, succ, val, full);
            const unsigned long long key = ((unsigned long long)n << 60) | (x << 6) | t;
            ha += sig_mix(key + 0x9E3779B97F4A7C15ull);
            hb += sig_mix(key * 0xD6E8FEB86659FD93ull + 0x2545F4914F6CDD1Dull);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        ha += __shfl_xor_sync(0xFFFFFFFFu, ha, o);
        hb += __shfl_xor_sync(0xFFFFFFFFu, hb, o);
    }
    if ((threadIdx.x & 31u) == 0) { s_a[threadIdx.x >> 5] = ha; s_b[threadIdx.x >> 5] = hb; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < 8; ++i) { ha += s_a[i]; hb += s_b[i]; }
        p.sig[2 * b] = ha;
        p.sig[2 * b + 1] = hb;
    }
}

}  // namespace

int launch_validity_bitmap(const ScanJob &job, uint32_t *bitmap_out, void *stream) {
    if (job.frame_count == 0 || job.n_formulas == 0) return 0;
    ValidityParams p;
    p.n = job.n; p.k = job.k; p.cls = job.cls; p.class_table = job.class_table;
    p.frame_begin = job.frame_begin; p.frame_count = job.frame_count;
    p.code = job.code; p.offsets = job.offsets; p.n_formulas = job.n_formulas;
    p.bitmap = bitmap_out; p.words = (job.frame_count + 31) / 32;
    const uint64_t bx = (job.frame_count + 127) / 128;
    if (bx > 0x7FFFFFFFull) return 801;
    // enough blocks to fill the device: split the formulas over blockIdx.y when the range is short
    const uint32_t by = (uint32_t)std::min<uint64_t>(job.n_formulas, std::max<uint64_t>(1, (148ull * 32 + bx - 1) / bx));
    validity_bitmap_kernel<<<dim3((uint32_t)bx, by), 128, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

int launch_condition_bitmap(uint32_t n, uint32_t cond, uint32_t cls, const uint64_t *class_table, uint64_t begin,
                            uint64_t count, uint32_t *bitmap_out, void *stream) {
    if (count == 0) return 0;
    ConditionParams p;
    p.n = n; p.cond = cond; p.cls = cls; p.class_table = class_table;
    p.frame_begin = begin; p.frame_count = count; p.bitmap = bitmap_out;
    const uint64_t bx = (count + 127) / 128;
    if (bx > 0x7FFFFFFFull) return 801;
    condition_bitmap_kernel<<<(uint32_t)bx, 128, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

int launch_frames_from_bitmap(uint32_t n, uint32_t cls, const uint64_t *class_table, uint64_t begin, uint64_t count,
                              const uint32_t *bitmap, uint16_t *succ_out, uint64_t capacity, uint64_t *count_out,
                              void *stream) {
    cudaError_t e = cudaMemsetAsync(count_out, 0, sizeof(uint64_t), (cudaStream_t)stream);
    if (e != cudaSuccess) return (int)e;
    if (count == 0) return 0;
    ConditionParams p;
    p.n = n; p.cond = 0; p.cls = cls; p.class_table = class_table;
    p.frame_begin = begin; p.frame_count = count; p.bitmap = const_cast<uint32_t *>(bitmap);
    const uint64_t bx = (count + 127) / 128;
    if (bx > 0x7FFFFFFFull) return 801;
    frames_from_bitmap_kernel<<<(uint32_t)bx, 128, 0, (cudaStream_t)stream>>>(
        p, succ_out, (unsigned long long)capacity, reinterpret_cast<unsigned long long *>(count_out));
    return (int)cudaGetLastError();
}

static int launch_density(const ScanJob &job, const uint16_t *succ_list, const uint32_t *records, uint32_t n_list,
                          const uint32_t *row_begin, const uint32_t *rows,
                          uint32_t *counts_out, uint64_t row_stride, uint64_t col_offset, void *stream) {
    if (job.frame_count == 0 || n_list == 0) return 0;
    DensityParams p;
    p.n = job.n; p.k = job.k; p.cls = job.cls; p.class_table = job.class_table; p.succ_list = succ_list;
    p.frame_begin = job.frame_begin; p.frame_count = job.frame_count;
    p.code = job.code; p.offsets = job.offsets; p.n_formulas = n_list; p.records = records; p.counts = counts_out;
    p.row_begin = row_begin; p.rows = rows;
    p.row_stride = row_stride; p.col_offset = col_offset;
    const uint64_t bx = (job.frame_count + 127) / 128;
    if (bx > 0x7FFFFFFFull) return 801;
    const uint32_t by = (uint32_t)std::min<uint64_t>(std::min<uint64_t>(n_list, 65535),
                                                     std::max<uint64_t>(1, (148ull * 32 + bx - 1) / bx));
    failure_density_kernel<<<dim3((uint32_t)bx, by), 128, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

int launch_failure_density(const ScanJob &job, const uint16_t *succ_list, uint32_t *counts_out, uint64_t row_stride,
                           uint64_t col_offset, void *stream) {
    return launch_density(job, succ_list, nullptr, job.n_formulas, nullptr, nullptr, counts_out, row_stride, col_offset, stream);
}

int launch_failure_density_records(const ScanJob &job, const uint32_t *records, uint32_t n_list, const uint32_t *row_begin,
                                   const uint32_t *rows, uint32_t *counts_out, uint64_t row_stride, uint64_t col_offset,
                                   void *stream) {
    return launch_density(job, nullptr, records, n_list, row_begin, rows, counts_out, row_stride, col_offset, stream);
}

int launch_match_bitmaps(const uint32_t *bitmaps, uint32_t n_records, uint64_t words, const uint32_t *library,
                         uint32_t n_library, uint32_t *match_out, void *stream) {
    if (n_records == 0) return 0;
    match_bitmaps_kernel<<<(n_records + 3) / 4, 128, 0, (cudaStream_t)stream>>>(bitmaps, n_records, words, library,
                                                                               n_library, match_out);
    return (int)cudaGetLastError();
}

int launch_signatures(uint32_t k, uint32_t n_max, const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                      uint64_t *sig_out, void *stream) {
    if (n_formulas == 0) return 0;
    SignatureParams p;
    p.k = k; p.n_max = n_max; p.code = code; p.offsets = offsets; p.n_formulas = n_formulas;
    p.sig = (unsigned long long *)sig_out;
    signature_kernel<<<n_formulas, 256, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

}  // namespace kripke
