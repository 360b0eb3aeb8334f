// adsc_resident3_d.cu — instantiations of the resident kernel (adsc_resident3.cuh): clusters of 3, 5 and 7 CTAs with the
// short segments (1024, 512, 256, 128 points), so that every N-1 = c * 2^k with c in {1, 3, 5, 7} and 2^k >= 128 up to
// 7168 has a resident configuration (N = 3073, 5121, 7169, 1537, ...).
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
#define ADSC_R3_ODD(P_, T_)                          \
    switch (cl) {                                    \
    case 3: ADSC_R3_KINDS(P_, T_, false, 3)          \
    case 5: ADSC_R3_KINDS(P_, T_, false, 5)          \
    case 7: ADSC_R3_KINDS(P_, T_, false, 7)          \
    default: return nullptr;                         \
    }

const void *res3_small_odd(int seg, int cl, int kind)
{
    switch (seg) {
    case 1024: ADSC_R3_ODD(8, 128)
    case 512: ADSC_R3_ODD(4, 128)
    case 256: ADSC_R3_ODD(4, 64)
    case 128: ADSC_R3_ODD(4, 32)
    default: return nullptr;
    }
}

}  // namespace adsc
