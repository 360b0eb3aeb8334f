// adsc_resident3_b.cu — instantiations of the resident kernel (adsc_resident3.cuh): clusters of 8 and 16 CTAs of 2048
// points (N-1 = 16384; 32768 = the paper's production grid), and the single-CTA configurations for
// short members (segments of 1024, 512, 256, 128 points).
#include "adsc_resident3.cuh"

namespace adsc {

#define ADSC_R3_KINDS(P_, T_, ACC_, CL_)                                                        \
    {                                                                                           \
        static const void *const f[4] = { (const void *)k_resident3<P_, T_, ACC_, CL_, false, 4>, \
                                          (const void *)k_resident3<P_, T_, ACC_, CL_, true, 4>,  \
                                          (const void *)k_resident3<P_, T_, ACC_, CL_, false, 3>, \
                                          (const void *)k_resident3<P_, T_, ACC_, CL_, false, 2> }; \
        return (kind >= 0 && kind < 4) ? f[kind] : nullptr;                                     \
    }

const void *res3_big_b(int cl, int kind)
{
    switch (cl) {
    case 8: ADSC_R3_KINDS(8, 256, true, 8)
    case 16: ADSC_R3_KINDS(8, 256, true, 16)
    default: return nullptr;
    }
}

const void *res3_small(int seg, int kind)
{
    switch (seg) {
    case 1024: ADSC_R3_KINDS(8, 128, false, 1)
    case 512: ADSC_R3_KINDS(4, 128, false, 1)
    case 256: ADSC_R3_KINDS(4, 64, false, 1)
    case 128: ADSC_R3_KINDS(4, 32, false, 1)
    default: return nullptr;
    }
}

}  // namespace adsc
