// kpz_launch_update_wide.cu -- one slice of the kernel instantiations of libkpz_b200.so (see kpz_host.h).
#include "kpz_launch.cuh"

int32_t kpz_launch_update_wide(kpz_ctx* c, const kpz::UpdateParams& P) {
    switch (c->T) {
        case 64: return kpz_launch::launch_update_mode<64, 96>(c, P);
        case 32: return kpz_launch::launch_update_mode<32, 64>(c, P);
    }
    return kpz_fail(c, KPZ_EINVAL, "unsupported tile %u", c->T);
}
