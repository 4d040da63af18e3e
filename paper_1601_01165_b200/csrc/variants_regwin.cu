// variants_regwin.cu -- KIND_REGWIN instantiations (fp32): register window reused across the
// thread's DMs.  TT = 12, 20, 28 make the LDS.128 window loads bank-conflict free (lane stride is
// an odd number of 16-byte chunks); RSTEP bounds the shift increment per DM step the switch covers.
#include "variants_common.cuh"

namespace dedisp {
#ifndef REGWIN_PART
#define REGWIN_PART 0
#endif
//                         In     kind       WD WT DT TT CC NS R  MINB
#if REGWIN_PART == 0
typedef Tile<float, KIND_REGWIN, 8, 1, 4, 28, 8, 3, 4, 1> R0;   // 32 x 896
typedef Tile<float, KIND_REGWIN, 4, 1, 4, 28, 8, 3, 4, 2> R1;   // 16 x 896
typedef Tile<float, KIND_REGWIN, 8, 1, 4, 20, 8, 3, 4, 1> R2;   // 32 x 640
void register_regwin0(std::vector<Variant> &r) {
    r.push_back(make_tiled<R0>());
    r.push_back(make_tiled<R1>());
    r.push_back(make_tiled<R2>());
}
#elif REGWIN_PART == 1
typedef Tile<float, KIND_REGWIN, 4, 2, 4, 20, 8, 3, 4, 1> R3;   // 16 x 1280
typedef Tile<float, KIND_REGWIN, 4, 1, 8, 12, 8, 3, 4, 2> R4;   // 32 x 384
typedef Tile<float, KIND_REGWIN, 4, 2, 6, 20, 8, 2, 4, 1> R5;   // 24 x 1280
void register_regwin1(std::vector<Variant> &r) {
    r.push_back(make_tiled<R3>());
    r.push_back(make_tiled<R4>());
    r.push_back(make_tiled<R5>());
}
#elif REGWIN_PART == 2
typedef Tile<float, KIND_REGWIN, 8, 1, 4, 12, 8, 3, 4, 2> R6;   // 32 x 384
typedef Tile<float, KIND_REGWIN, 4, 2, 4, 16, 8, 3, 4, 2> R7;   // 16 x 1024 (conflicting stride)
typedef Tile<float, KIND_REGWIN, 4, 1, 2, 28, 8, 3, 4, 3> R8;   // 8 x 896
void register_regwin2(std::vector<Variant> &r) {
    r.push_back(make_tiled<R6>());
    r.push_back(make_tiled<R7>());
    r.push_back(make_tiled<R8>());
}
#else
typedef Tile<float, KIND_REGWIN, 4, 2, 8, 12, 8, 2, 4, 1> R9;   // 32 x 768
typedef Tile<float, KIND_REGWIN, 4, 1, 4, 28, 8, 3, 6, 2> R10;  // 16 x 896, r6
typedef Tile<float, KIND_REGWIN, 2, 2, 4, 12, 8, 2, 2, 3> R11;  // 8 x 768, r2
void register_regwin3(std::vector<Variant> &r) {
    r.push_back(make_tiled<R9>());
    r.push_back(make_tiled<R10>());
    r.push_back(make_tiled<R11>());
}
#endif
}  // namespace dedisp
