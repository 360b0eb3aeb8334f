// adsc_resident3_a.cu — instantiations of the resident kernel (adsc_resident3.cuh): 8 points per thread, 256 threads
// (2048-point segments), clusters of 1, 2 and 4 CTAs per member (N-1 = 2048, 4096, 8192: BASELINE.json configs[4], [1], [2]).
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

const void *res3_big_a(int cl, int kind)
{
    switch (cl) {
    case 1: ADSC_R3_KINDS(8, 256, true, 1)
    case 2: ADSC_R3_KINDS(8, 256, true, 2)
    case 4: ADSC_R3_KINDS(8, 256, true, 4)
    default: return nullptr;
    }
}

}  // namespace adsc
