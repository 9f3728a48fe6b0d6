// internal.h - declarations shared by the host translation units of libkripke_b200.so.
#pragma once
#include <stdint.h>

#include <vector>

#include "../../include/kripke.h"
#include "ucode.h"

namespace kripke {

// ---- lower.cpp ---------------------------------------------------------------------------------
struct Lowered {
    std::vector<uint16_t> ucode;  // micro-ops (op | arg << 8), FIN last
    int need = 0;                 // register-stack slots needed (fits the sliced kernel iff <= UC_DMAX)
    uint32_t n_modal = 0;         // executed box/dia micro-ops
    uint32_t n_bool = 0;          // executed and/or/andn/nand micro-ops
};
int validate_programs(const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas, uint32_t n_vars,
                      uint32_t *max_stack_out);
// Variables a program still mentions after constant folding (bit i = p_i).
uint32_t program_support(const uint8_t *code, uint32_t len);
// rename: variable index -> index in the reduced valuation (null = identity).
bool lower_single(const uint8_t *code, uint32_t len, uint32_t mode, const uint8_t *rename, Lowered *out);
bool lower_pair(const uint8_t *code_a, uint32_t len_a, const uint8_t *code_b, uint32_t len_b, uint32_t mode,
                const uint8_t *rename, Lowered *out);

// ---- device-side job description (kernels) -----------------------------------------------------
// Accumulators per output record, owned by the programs handle, zeroed at the start of a call.
struct Accum {
    unsigned long long models;
    unsigned long long frames;
    unsigned long long best;      // least class-frame index (or unit) with a hit; ~0 = none
};

struct ScanJob {
    // what to scan
    uint32_t n;                   // worlds
    uint32_t k;                   // variables
    uint32_t cls;                 // frame class
    uint64_t frame_begin;         // class-order range
    uint64_t frame_count;
    const uint64_t *class_table;  // device: ascending K-indices for S4 / S5 (else null)
    // programs (raw postfix form; used by the scalar kernel and by witness completion)
    const uint8_t *code;          // device
    const uint32_t *offsets;      // device, n_formulas + 1
    uint32_t n_formulas;
    // records: either one per formula (pairs == null) or one per pair
    const uint32_t *pairs;        // device, 2 * n_records, or null
    uint32_t n_records;
    Accum *accum;                 // device, n_records
};

// ---- launch wrappers (defined in the .cu files) ------------------------------------------------
struct SlicedPlan {
    // lowered slots (a slot is one record the sliced kernel evaluates)
    const uint16_t *ucode;        // device: n_slots * stride micro-ops
    const uint32_t *slot_record;  // device: record index per slot
    uint32_t n_slots;
    uint32_t stride;              // micro-ops per slot (even, >= longest program + 1)
    uint32_t max_need;            // most register-stack slots any slot needs
    uint32_t model_shift;         // refuting models are counted x 2^model_shift (unused variables)
};

// Is there a sliced instantiation for this shape and class that keeps `need` stack slots?  If so
// *frames_per_unit is the alignment frame ranges must have for it.
bool sliced_select(uint32_t n, uint32_t k, uint32_t cls, uint32_t need, uint64_t *frames_per_unit);
// Index of the instantiation `sliced_select` would pick (UINT32_MAX = none).
uint32_t sliced_row(uint32_t n, uint32_t k, uint32_t cls, uint32_t need);
// LOWER_* flags for the instantiations this shape and class run on (0 = no shape): classes other than K
// can only use the frame-per-unit rows, whose derived leaves differ from the group-per-unit rows'.
uint32_t sliced_lower_mode(uint32_t n, uint32_t k, uint32_t cls);
// Should programs of this need class be lowered with LOWER_FUSE?
bool sliced_fuses(uint32_t n, uint32_t k, uint32_t need);
// Enqueue the sliced scan; returns a cudaError_t as int and the number of kernel launches.
int launch_sliced(const ScanJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches);
// Enqueue the scalar (Algorithm 1) scan over the records listed in `records` (device, or null = all).
int launch_scalar(const ScanJob &job, const uint32_t *records, uint32_t n_list, uint32_t reduce_mode,
                  void *stream, uint32_t *launches);
// ---- frame-list mode (scan_frames.cu) ----------------------------------------------------------
struct FramesJob {
    uint32_t n, k;
    const uint16_t *succ;         // device: n_frames * n successor masks
    uint64_t n_frames;
    uint64_t index_base;          // added to the list position in witness.frame
    const uint8_t *code;          // device (raw postfix form: scalar kernel, witness completion)
    const uint32_t *offsets;
    const uint32_t *pairs;        // device, 2 * n_records, or null
    uint32_t n_records;
    Accum *accum;
};
// Bit-sliced scan of the lowered slots over the list (32 frames per word); n <= 16.
int launch_frames(const FramesJob &job, const SlicedPlan &plan, void *stream, uint32_t *launches);
// Scalar scan (thread = frame) of the listed records (device list, or null = all).
int launch_frames_scalar(const FramesJob &job, const uint32_t *records, uint32_t n_list, void *stream,
                         uint32_t *launches);
int launch_frames_finish(const FramesJob &job, bool accumulate, kripke_count_t *counts_out,
                         kripke_witness_t *witness_out, void *stream);

// ---- correspondence recovery (bitmaps.cu) ------------------------------------------------------
int launch_validity_bitmap(const ScanJob &job, uint32_t *bitmap_out, void *stream);
int launch_condition_bitmap(uint32_t n, uint32_t cond, uint32_t cls, const uint64_t *class_table, uint64_t begin,
                            uint64_t count, uint32_t *bitmap_out, void *stream);
int launch_frames_from_bitmap(uint32_t n, uint32_t cls, const uint64_t *class_table, uint64_t begin, uint64_t count,
                              const uint32_t *bitmap, uint16_t *succ_out, uint64_t capacity, uint64_t *count_out,
                              void *stream);
// Failure densities: frames of job's class range, or of succ_list (job.frame_count masks rows) if not null.
// counts_out[record * row_stride + col_offset + j] for frame j of the job's range (all formulas, or the listed records).
int launch_failure_density(const ScanJob &job, const uint16_t *succ_list, uint32_t *counts_out, uint64_t row_stride,
                           uint64_t col_offset, void *stream);
// records[i] is evaluated once and written to the rows rows[row_begin[i] .. row_begin[i+1]) (row tables null: to its own row)
int launch_failure_density_records(const ScanJob &job, const uint32_t *records, uint32_t n_list, const uint32_t *row_begin,
                                   const uint32_t *rows, uint32_t *counts_out, uint64_t row_stride, uint64_t col_offset,
                                   void *stream);
int launch_match_bitmaps(const uint32_t *bitmaps, uint32_t n_records, uint64_t words, const uint32_t *library,
                         uint32_t n_library, uint32_t *match_out, void *stream);

// Frame-list generators (frame_gen.cu): n_frames x n successor masks written on the device.
int launch_frames_generate(uint32_t gen, uint32_t n, uint64_t n_frames, uint64_t seed, uint16_t *succ_out, void *stream);

// Semantic signatures: two 64-bit sums per formula over every model of 1..n_max worlds.
int launch_signatures(uint32_t k, uint32_t n_max, const uint8_t *code, const uint32_t *offsets, uint32_t n_formulas,
                      uint64_t *sig_out, void *stream);

// Zero the accumulators; finish: turn accumulators into counts / witnesses (handles ACCUMULATE).
int launch_init(Accum *accum, uint32_t n_records, void *stream);
// accum[pairs[2i]] = accum[pairs[2i+1]] for i < n (records sharing a representative's program).
int launch_alias_accum(Accum *accum, const uint32_t *pairs, uint32_t n, void *stream);
int launch_finish(const ScanJob &job, bool accumulate, kripke_count_t *counts_out,
                  kripke_witness_t *witness_out, void *stream);
// Size record of step H8.
int launch_record_size(uint32_t n, uint32_t n_records, const kripke_count_t *cnt, const kripke_witness_t *wit,
                       uint32_t *size_out, kripke_count_t *counts_out, kripke_witness_t *witness_out, void *stream);
// Witness records <-> 64-bit keys (multi-GPU exchange step).
int launch_witness_keys(bool to_keys, const void *src, uint32_t n_records, uint32_t kn, void *dst, void *stream);
// Calibration kernels.
int run_calibration(uint32_t variant, double *rate_out, double *ms_out, void *stream);

// ---- error bookkeeping (api.cpp) ---------------------------------------------------------------
// Stores e (a cudaError_t) as this thread's last CUDA error and returns KRIPKE_ECUDA.
int note_cuda_error(int e);

// ---- class tables (api.cpp) --------------------------------------------------------------------
// Host: ascending K-indices of the class members (S4 / S5), n <= 5 here; cached.
const std::vector<uint64_t> *class_table_host(uint32_t n, uint32_t cls);

}  // namespace kripke
