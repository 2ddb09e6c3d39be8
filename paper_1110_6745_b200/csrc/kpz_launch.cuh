// kpz_launch.cuh -- launch templates of the update kernels, included by the kpz_launch_*.cu translation units.
#pragma once
#include "kpz_host.h"

namespace kpz_launch {

template <int T, int NTHR, int MODE, bool DEAD, int SUB>
int32_t launch_update_k(kpz_ctx* c, const kpz::UpdateParams& P) {
    const size_t smem = (size_t)kpz::TileGeom<T>::WORDS * NTHR * sizeof(uint32_t);
    auto kern = kpz::kpz_update_kernel<T, NTHR, MODE, DEAD, SUB>;
    // function attributes are per device: one flag per device ordinal and instantiation
    static bool attr_set[KPZ_MAX_DEVICES] = {};
    const int dev = (c->device >= 0 && c->device < KPZ_MAX_DEVICES) ? c->device : 0;
    if (!attr_set[dev]) {
        KPZ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        KPZ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        attr_set[dev] = true;
    }
    const uint64_t blocks = (P.total_items + NTHR - 1) / NTHR;
    if (blocks > 0x7FFFFFFFull) return kpz_fail(c, KPZ_EINVAL, "too many tiles for one launch");
    kern<<<(unsigned)blocks, NTHR, smem, c->stream>>>(P);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches++;
    return KPZ_OK;
}

template <int T, int NTHR, int MODE, bool DEAD>
int32_t launch_update_t(kpz_ctx* c, const kpz::UpdateParams& P) {
    if (c->poisson) return launch_update_k<T, NTHR, MODE, DEAD, 2>(c, P);
    return c->sub_sweeps > 1 ? launch_update_k<T, NTHR, MODE, DEAD, 1>(c, P) : launch_update_k<T, NTHR, MODE, DEAD, 0>(c, P);
}

template <int T, int NTHR, bool DEAD>
int32_t launch_update_sched(kpz_ctx* c, const kpz::UpdateParams& P) {
    if (c->p >= 1.0 && c->q <= 0.0) return launch_update_t<T, NTHR, 0, DEAD>(c, P);
    if (P.thr_p >= 1 && P.thr_q >= 1) return launch_update_t<T, NTHR, 1, DEAD>(c, P);
    return launch_update_t<T, NTHR, 2, DEAD>(c, P);
}

template <int T, int NTHR>
int32_t launch_update_mode(kpz_ctx* c, const kpz::UpdateParams& P) {
    return c->schedule == KPZ_SCHEDULE_DEAD_BORDER ? launch_update_sched<T, NTHR, true>(c, P)
                                                   : launch_update_sched<T, NTHR, false>(c, P);
}

template <int T, int NTHR, int MODE>
int32_t launch_resident_k(kpz_ctx* c, const kpz::UpdateParams& P, const ResidentPlan& pl, uint32_t n_mcs) {
    auto kern = kpz::kpz_resident_kernel<T, NTHR, MODE>;
    static bool attr_set[KPZ_MAX_DEVICES] = {};
    const int dev = (c->device >= 0 && c->device < KPZ_MAX_DEVICES) ? c->device : 0;
    if (!attr_set[dev]) {
        KPZ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)KPZ_RESIDENT_SMEM_MAX));
        attr_set[dev] = true;
    }
    kern<<<pl.blocks, NTHR, pl.smem, c->stream>>>(P, pl.G, n_mcs, c->R, c->sub_sweeps);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches++;
    return KPZ_OK;
}

template <int T, int NTHR>
int32_t launch_resident_m(kpz_ctx* c, const kpz::UpdateParams& P, const ResidentPlan& pl, uint32_t n_mcs) {
    if (c->p >= 1.0 && c->q <= 0.0) return launch_resident_k<T, NTHR, 0>(c, P, pl, n_mcs);
    if (P.thr_p >= 1 && P.thr_q >= 1) return launch_resident_k<T, NTHR, 1>(c, P, pl, n_mcs);
    return launch_resident_k<T, NTHR, 2>(c, P, pl, n_mcs);
}

template <int T>
int32_t launch_resident_t(kpz_ctx* c, const kpz::UpdateParams& P, const ResidentPlan& pl, uint32_t n_mcs) {
    switch (pl.nthr) {
        case 256: return launch_resident_m<T, 256>(c, P, pl, n_mcs);
        case 128: return launch_resident_m<T, 128>(c, P, pl, n_mcs);
        case 64: return launch_resident_m<T, 64>(c, P, pl, n_mcs);
        default: return launch_resident_m<T, 32>(c, P, pl, n_mcs);
    }
}


}  // namespace kpz_launch
