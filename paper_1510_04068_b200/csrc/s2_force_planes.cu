// s2_force_planes.cu -- how many 16-byte planes a force kernel variant stages per j tile.
#include "s2_internal.h"

namespace s2 {

int force_nplanes(int precision, int order, unsigned flags)
{
    const int dec = flags ? 2 : 0;   // fp64 position planes for the nn / neighbour decisions
    switch (precision) {
    case S2_FP64: return order == 6 ? 6 : (order == 2 ? 3 : 4);
    case S2_FP32: return (order == 6 ? 4 : (order == 2 ? 2 : 3)) + dec;
    case S2_DS: return (order == 6 ? 6 : (order == 2 ? 3 : 4)) + dec;
    }
    return 0;
}

}  // namespace s2
