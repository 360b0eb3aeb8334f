// adsc_resident3_e.cu — instantiations of the resident kernel (adsc_resident3.cuh): clusters of 2, 4 and 8 CTAs of the
// short segments (1024, 512, 256 points).  The default selection never takes them (a wider segment tiles the same N);
// ADSC_OPT_SPREAD does, to put more SMs on each member of an ensemble that does not fill the device.
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
#define ADSC_R3_EVEN(P_, T_)                         \
    switch (cl) {                                    \
    case 2: ADSC_R3_KINDS(P_, T_, false, 2)          \
    case 4: ADSC_R3_KINDS(P_, T_, false, 4)          \
    case 8: ADSC_R3_KINDS(P_, T_, false, 8)          \
    default: return nullptr;                         \
    }

const void *res3_small_even(int seg, int cl, int kind)
{
    switch (seg) {
    case 1024: ADSC_R3_EVEN(8, 128)
    case 512: ADSC_R3_EVEN(4, 128)
    case 256: ADSC_R3_EVEN(4, 64)
    default: return nullptr;
    }
}

}  // namespace adsc
