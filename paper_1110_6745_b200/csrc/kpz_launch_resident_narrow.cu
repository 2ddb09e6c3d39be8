// kpz_launch_resident_narrow.cu -- one slice of the kernel instantiations of libkpz_b200.so (see kpz_host.h).
#include "kpz_launch.cuh"

int32_t kpz_launch_resident_narrow(kpz_ctx* c, const kpz::UpdateParams& P, const ResidentPlan& pl, uint32_t n_mcs) {
    switch (c->T) {
        case 16: return kpz_launch::launch_resident_t<16>(c, P, pl, n_mcs);
        case 8: return kpz_launch::launch_resident_t<8>(c, P, pl, n_mcs);
        case 4: return kpz_launch::launch_resident_t<4>(c, P, pl, n_mcs);
    }
    return kpz_fail(c, KPZ_EINVAL, "unsupported tile %u", c->T);
}
