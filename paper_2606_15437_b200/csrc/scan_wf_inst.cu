// scan_wf_inst.cu - instantiations, launcher and cost model of the warp-frame kernel (scan_wf.cuh).
#include <memory>

#include "scan_wf.cuh"

namespace kripke {

namespace {

// Expected logic instructions for one result word of row w (average over the class: every
// compile-time and uniform edge bit is present in exactly half of the frames): a data edge costs one
// 3-input instruction; s set edges cost ceil(s/2) on top of a running value, ceil((s-1)/2) alone.
template <class C>
double row_cost(int w) {
    int nd = 0, na = 0, nfree = 0;
    for (int u = 0; u < C::N; ++u) {
        const int c = C::edge_class(w, u);
        if (c == EC_WORD || c == EC_LANE) ++nd;
        else if (c == EC_ALWAYS) ++na;
        else ++nfree;
    }
    double sum = 0;
    for (int sub = 0; sub < (1 << nfree); ++sub) {
        const int s = na + __builtin_popcount(sub);
        sum += nd + (nd > 0 ? (s + 1) / 2 : (s > 0 ? s / 2 : 0));
    }
    return sum / (1 << nfree);
}

template <class C>
double cost_per_frame(const WfOpCounts &c) {
    const int N = C::N, M = C::M;
    double modal_s = 0, modal_f = 0;
    for (int w = 0; w < N; ++w) {
        modal_s += row_cost<C>(w) * (w == C::W0 ? M : 1);
        modal_f += row_cost<C>(w) * M;
    }
    const double fin_word = (N - 1 + 1) / 2 + 2;               // AND of n words, popc, add
    const double fin[3] = {fin_word, (double)((N - 2 + 1) / 2) + 3.0 * M, fin_word * M};
    const double per_unit = c.bool_s * N + c.bool_h * (N - 1 + M) + c.bool_f * (M * N) + c.modal_s * modal_s +
                            c.modal_hf * modal_f + fin[c.fin_type < 3 ? c.fin_type : 2];
    return per_unit * 32.0 / (double)(1ull << C::UFB);         // 32 lanes execute it; 2^UFB frames per unit
}

template <class C, int MINB>
int launch_wf_inst(const ScanJob &job, const WfPlan &plan, void *stream, uint32_t *launches) {
    static int grid_full = 0;
    auto kern = scan_wf_kernel<C, MINB>;
    if (!grid_full) {
        int dev = 0, sms = 0, b = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return (int)e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, kern, 32, 0);
        if (e != cudaSuccess) return (int)e;
        grid_full = sms * (b > 0 ? b : 1);
    }
    const uint64_t unit_begin = job.frame_begin >> C::UFB, unit_count = job.frame_count >> C::UFB;
    if (unit_count == 0 || plan.n_progs == 0) return 0;
    std::unique_ptr<WfParams> prm(new WfParams);
    uint32_t p0 = 0;
    while (p0 < plan.n_progs) {
        // as many programs as fit the parameter block
        uint32_t p1 = p0;
        const uint32_t base = plan.prog_off[p0];
        while (p1 < plan.n_progs && p1 - p0 < WF_MAX_PROGS && plan.prog_off[p1 + 1] - base <= WF_MAX_UCODE) ++p1;
        if (p1 == p0) return (int)cudaErrorInvalidValue;        // one program longer than the block
        WfParams &q = *prm;
        q.unit_begin = unit_begin;
        q.unit_count = unit_count;
        q.n_progs = p1 - p0;
        q.model_shift = plan.model_shift;
        q.accum = job.accum;
        q.prog_record = plan.prog_record + p0;
        for (uint32_t i = p0; i <= p1; ++i) q.prog_off[i - p0] = (uint16_t)(plan.prog_off[i] - base);
        std::copy(plan.ucode.begin() + base, plan.ucode.begin() + plan.prog_off[p1], q.ucode);
        // work items: enough to balance the grid, each long enough to amortise its atomics
        uint64_t upi = unit_count * q.n_progs / ((uint64_t)grid_full * 16);
        upi = std::max<uint64_t>(1, std::min<uint64_t>(upi, 2048));
        upi = std::min<uint64_t>(upi, unit_count);
        q.units_per_item = (uint32_t)upi;
        q.n_ranges = (uint32_t)((unit_count + upi - 1) / upi);
        const uint64_t items = (uint64_t)q.n_ranges * q.n_progs;
        const uint32_t grid = (uint32_t)std::min<uint64_t>(items, (uint64_t)grid_full);
        kern<<<grid, 32, 0, (cudaStream_t)stream>>>(q);
        if (launches) ++*launches;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return (int)e;
        p0 = p1;
    }
    return 0;
}

}  // namespace

// One instantiation per translation unit (they compile in parallel): -DKRIPKE_WF_INST=<0..4>.
// Keep in step with wf_dispatch.cpp.  WF_INST(index, n, k, MB, class, MINB): M = 2^MB sibling frames
// per thread, MINB resident one-warp blocks per SM (register budget 65536 / (32 * MINB)).
#define WF_INST(IDX, N, K, MB, CLS, MINB)                                                          \
    extern const WfRow kWfRow##IDX = {N, K, CLS, 1ull << WfCfg<N, K, MB, CLS>::UFB,                \
                                      launch_wf_inst<WfCfg<N, K, MB, CLS>, MINB>,                  \
                                      cost_per_frame<WfCfg<N, K, MB, CLS>>};

#ifndef KRIPKE_WF_INST
#error "compile with -DKRIPKE_WF_INST=<0..4>"
#elif KRIPKE_WF_INST == 0
WF_INST(0, 5, 2, 3, KRIPKE_CLASS_K, 8)
#elif KRIPKE_WF_INST == 1
WF_INST(1, 5, 1, 3, KRIPKE_CLASS_K, 8)
#elif KRIPKE_WF_INST == 2
WF_INST(2, 5, 0, 3, KRIPKE_CLASS_K, 12)
#elif KRIPKE_WF_INST == 3
WF_INST(3, 5, 2, 3, KRIPKE_CLASS_T, 8)
#elif KRIPKE_WF_INST == 4
WF_INST(4, 5, 1, 3, KRIPKE_CLASS_T, 8)
#endif

}  // namespace kripke
