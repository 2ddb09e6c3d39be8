// kpz_launch_update_narrow.cu -- one slice of the kernel instantiations of libkpz_b200.so (see kpz_host.h).
#include "kpz_launch.cuh"

int32_t kpz_launch_update_narrow(kpz_ctx* c, const kpz::UpdateParams& P) {
    switch (c->T) {
        case 16: return kpz_launch::launch_update_mode<16, 128>(c, P);
        case 8: return kpz_launch::launch_update_mode<8, 128>(c, P);
        case 4: return kpz_launch::launch_update_mode<4, 128>(c, P);
    }
    return kpz_fail(c, KPZ_EINVAL, "unsupported tile %u", c->T);
}
