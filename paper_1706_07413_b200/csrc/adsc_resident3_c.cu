// adsc_resident3_c.cu — instantiations of the resident kernel (adsc_resident3.cuh): clusters of 3, 5, 6 and 7 CTAs of
// 2048 points (N-1 = 6144, 10240, 12288, 14336).
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

const void *res3_big_c(int cl, int kind)
{
    switch (cl) {
    case 3: ADSC_R3_KINDS(8, 256, true, 3)
    case 5: ADSC_R3_KINDS(8, 256, true, 5)
    case 6: ADSC_R3_KINDS(8, 256, true, 6)
    case 7: ADSC_R3_KINDS(8, 256, true, 7)
    default: return nullptr;
    }
}

}  // namespace adsc
