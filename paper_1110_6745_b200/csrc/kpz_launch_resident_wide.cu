// kpz_launch_resident_wide.cu -- one slice of the kernel instantiations of libkpz_b200.so (see kpz_host.h).
#include "kpz_launch.cuh"

int32_t kpz_launch_resident_wide(kpz_ctx* c, const kpz::UpdateParams& P, const ResidentPlan& pl, uint32_t n_mcs) {
    switch (c->T) {
        case 64: return kpz_launch::launch_resident_t<64>(c, P, pl, n_mcs);
        case 32: return kpz_launch::launch_resident_t<32>(c, P, pl, n_mcs);
    }
    return kpz_fail(c, KPZ_EINVAL, "unsupported tile %u", c->T);
}
