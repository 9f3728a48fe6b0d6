// scan_static.cu - kripke_eval_batch_static: the scalar corpus scan (Algorithm 1) for callers
// that must not allocate device memory.
//
// Who this is for.  Every other scan of this library goes through a kripke_programs_t handle, and creating or
// using a handle calls cudaMalloc (device copies of the programs, the per-record accumulators, the S4 / S5 class
// table; the compiled engine also loads freshly built modules).  Some users cannot afford that:
//   - a process whose device memory already belongs to somebody else's pool (a torch process whose caching
//     allocator was given the whole card, an inference server that reserved its HBM at start-up): a cudaMalloc
//     there fails, or takes memory behind the pool's back;
//   - a latency-sensitive loop with other streams in flight: cudaMalloc and cudaFree synchronise the whole
//     device, so an allocation inside a call stalls work that has nothing to do with it.
// For them this file keeps everything the scan needs beyond the caller's own buffers in ONE fixed block of device
// memory that is part of the library image (g_static_scratch below).  The entry point calls no cudaMalloc, no
// cudaFree and no library routine that allocates; it only copies the (host) programs into the block and enqueues
// the scalar kernels of scan_scalar.cu on it.
//
// What it costs.  KRIPKE_STATIC_SCRATCH_BYTES (about 0.8 MB) of device memory on every GPU on which the library
// is loaded, from load until the process exits, whether or not this entry point is ever called; and fixed
// limits (KRIPKE_STATIC_MAX_FORMULAS, KRIPKE_STATIC_MAX_CLASS_FRAMES) instead of "whatever fits".
//
// The block is shared by all calls.  It keeps what the previous call left in it, so every call re-initialises
// the part it reads before writing (the accumulators; programs, offsets and class table are overwritten up to
// the lengths the kernels read).  Two calls whose device work overlaps - different streams without an event
// between them, or different host threads - use the same accumulators and program bytes at the same time and
// corrupt each other: serialise them on one stream or with events.
#include <cuda_runtime.h>

#include <cstddef>
#include <mutex>

#include "internal.h"

namespace {

using kripke::Accum;

// Layout of the block; every section starts on a 256-byte boundary.
constexpr size_t up256(size_t x) { return (x + 255) / 256 * 256; }
constexpr size_t OFF_ACCUM = 0;
constexpr size_t OFF_TABLE = up256(OFF_ACCUM + sizeof(Accum) * KRIPKE_STATIC_MAX_FORMULAS);
constexpr size_t OFF_OFFSETS = up256(OFF_TABLE + sizeof(uint64_t) * KRIPKE_STATIC_MAX_CLASS_FRAMES);
constexpr size_t OFF_CODE = up256(OFF_OFFSETS + sizeof(uint32_t) * (KRIPKE_STATIC_MAX_FORMULAS + 1));
constexpr size_t SCRATCH_BYTES = up256(OFF_CODE + (size_t)KRIPKE_STATIC_MAX_FORMULAS * KRIPKE_MAX_PROGRAM_LEN);
static_assert(SCRATCH_BYTES == KRIPKE_STATIC_SCRATCH_BYTES, "include/kripke.h states the size of the static block");

// The block.  In HOST code this name is only a handle for the runtime's symbol calls - it is not a device
// address, and a kernel handed `g_static_scratch` from the host would fault or scribble over unrelated memory.
// The address the kernels get is the one cudaGetSymbolAddress returns (scratch_for_current_device below).
static __device__ __align__(256) unsigned char g_static_scratch[SCRATCH_BYTES];

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
unsigned char *g_scratch_ptr[MAX_DEVICES] = {};   // per device ordinal; filled on the first call on that device

// Set-up, once per device, with that device current: ask the runtime where this device's copy of the block is.
int scratch_for_current_device(unsigned char **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return kripke::note_cuda_error((int)e);
    if (dev < 0 || dev >= MAX_DEVICES) return KRIPKE_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return kripke::note_cuda_error((int)e);
        if (!p) return kripke::note_cuda_error((int)cudaErrorInvalidSymbol);
        g_scratch_ptr[dev] = (unsigned char *)p;
    }
    *out = g_scratch_ptr[dev];
    return KRIPKE_OK;
}

constexpr uint32_t STATIC_FLAGS = KRIPKE_ACCUMULATE | KRIPKE_REDUCE_MASK;

}  // namespace

extern "C" int kripke_eval_batch_static(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                                        uint32_t n_worlds, uint32_t n_vars, uint32_t frame_class,
                                        uint64_t frame_begin, uint64_t frame_count, uint32_t flags,
                                        kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream) {
    using namespace kripke;
    // ---- host-only checks first: nothing below this block is reached with sizes the static block cannot hold
    if (!offsets || (n_formulas && !code)) return KRIPKE_EINVAL;
    if (n_formulas && (!counts_out || !witness_out)) return KRIPKE_EINVAL;
    if (flags & ~STATIC_FLAGS) return KRIPKE_EINVAL;
    const uint32_t reduce = (flags & KRIPKE_REDUCE_MASK) >> 8;
    if (reduce > 2) return KRIPKE_EINVAL;
    if (n_worlds < 1 || n_worlds > KRIPKE_MAX_WORLDS || n_vars > KRIPKE_MAX_VARS || frame_class > KRIPKE_CLASS_S5)
        return KRIPKE_EINVAL;
    if (n_worlds * n_worlds + n_vars * n_worlds > KRIPKE_MAX_MODEL_BITS) return KRIPKE_EUNSUPPORTED;
    if (n_formulas > KRIPKE_STATIC_MAX_FORMULAS) return KRIPKE_EUNSUPPORTED;          // the batch limit
    const bool tabled = frame_class == KRIPKE_CLASS_S4 || frame_class == KRIPKE_CLASS_S5;
    if (tabled && n_worlds > 5) return KRIPKE_EUNSUPPORTED;                           // 209,527 preorders: no room
    uint64_t csize = 0;
    int rc = kripke_class_size(n_worlds, frame_class, &csize);
    if (rc) return rc;
    if (tabled && csize > KRIPKE_STATIC_MAX_CLASS_FRAMES) return KRIPKE_EUNSUPPORTED; // the class-table limit
    if (frame_begin > csize || frame_count > csize - frame_begin) return KRIPKE_EINVAL;
    if ((rc = validate_programs(code, offsets, n_formulas, n_vars, nullptr))) return rc;
    const uint32_t code_begin = offsets[0], code_bytes = offsets[n_formulas] - offsets[0];
    // (validate_programs bounds every program by KRIPKE_MAX_PROGRAM_LEN, so code_bytes fits its section)
    if (n_formulas == 0) return KRIPKE_OK;

    // ---- set-up (first call on this device) and the device addresses of the sections
    unsigned char *base = nullptr;
    if ((rc = scratch_for_current_device(&base))) return rc;
    Accum *d_accum = (Accum *)(base + OFF_ACCUM);
    uint64_t *d_table = (uint64_t *)(base + OFF_TABLE);
    uint32_t *d_offsets = (uint32_t *)(base + OFF_OFFSETS);
    uint8_t *d_code = base + OFF_CODE;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;

    // ---- inputs into the block, in stream order behind whatever the previous call on this stream left running.
    // The code section receives code[offsets[0] .. offsets[B]); the offsets are copied as given.
    if (code_bytes &&
        (e = cudaMemcpyAsync(d_code, code + code_begin, code_bytes, cudaMemcpyHostToDevice, s)) != cudaSuccess)
        return note_cuda_error((int)e);
    if ((e = cudaMemcpyAsync(d_offsets, offsets, sizeof(uint32_t) * ((size_t)n_formulas + 1), cudaMemcpyHostToDevice,
                             s)) != cudaSuccess)
        return note_cuda_error((int)e);
    if (tabled) {
        const std::vector<uint64_t> *t = class_table_host(n_worlds, frame_class);   // cached for the process
        if (t->size() != csize) return KRIPKE_EINVAL;
        if (csize && (e = cudaMemcpyAsync(d_table, t->data(), sizeof(uint64_t) * csize, cudaMemcpyHostToDevice, s)) !=
                         cudaSuccess)
            return note_cuda_error((int)e);
    }

    // ---- the scan itself: the kernels of scan_scalar.cu, unchanged, with the block as their scratch
    ScanJob job;
    job.n = n_worlds; job.k = n_vars; job.cls = frame_class;
    job.frame_begin = frame_begin; job.frame_count = frame_count;
    job.class_table = tabled ? d_table : nullptr;
    // the kernels read program b at job.code + offsets[b], and every offsets[b] >= offsets[0]: shift the base so
    // that the caller's offsets land in the code section (the shifted address itself is never dereferenced)
    job.code = (const uint8_t *)((uintptr_t)d_code - (uintptr_t)code_begin);
    job.offsets = d_offsets;
    job.n_formulas = n_formulas;
    job.pairs = nullptr;
    job.n_records = n_formulas;
    job.accum = d_accum;
    int ce;
    if ((ce = launch_init(d_accum, n_formulas, stream))) return note_cuda_error(ce);   // what must start at zero
    if ((ce = launch_scalar(job, nullptr, n_formulas, reduce, stream, nullptr))) return note_cuda_error(ce);
    if ((ce = launch_finish(job, (flags & KRIPKE_ACCUMULATE) != 0, counts_out, witness_out, stream)))
        return note_cuda_error(ce);
    return KRIPKE_OK;
}
