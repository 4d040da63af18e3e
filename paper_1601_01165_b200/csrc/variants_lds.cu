// variants_lds.cu -- KIND_LDS instantiations (fp32): staged tile, one shared-memory word per add.
// These run any setup (no limit on the shift increment per DM step), e.g. the LOFAR-like one.
#include "variants_common.cuh"

namespace dedisp {
//                      In     kind     WD WT DT TT CC NS R  MINB
typedef Tile<float, KIND_LDS, 4, 2, 4, 4, 8, 3, 0, 2> L0;   // 16 x 256
typedef Tile<float, KIND_LDS, 8, 1, 4, 8, 8, 3, 0, 2> L1;   // 32 x 256
typedef Tile<float, KIND_LDS, 4, 2, 8, 4, 8, 3, 0, 2> L2;   // 32 x 256
typedef Tile<float, KIND_LDS, 4, 2, 4, 8, 8, 2, 0, 2> L3;   // 16 x 512
typedef Tile<float, KIND_LDS, 2, 4, 4, 8, 8, 2, 0, 2> L4;   // 8 x 1024
typedef Tile<float, KIND_LDS, 2, 4, 8, 4, 16, 2, 0, 2> L5;  // 16 x 512, deeper chunk
typedef Tile<float, KIND_LDS, 2, 2, 2, 2, 8, 2, 0, 4> L6;   // 4 x 128 (small problems)
typedef Tile<float, KIND_LDS, 1, 8, 8, 4, 16, 2, 0, 2> L7;  // 8 x 1024
typedef Tile<float, KIND_LDS, 2, 4, 8, 8, 16, 2, 0, 1> L8;  // 16 x 1024
// long shifts (the paper's LOFAR setup, DM step 0.25: up to ~900 samples per DM step): few channels per
// stage so that the long spans of a DM tile still fit shared memory
typedef Tile<float, KIND_LDS, 1, 8, 4, 8, 2, 3, 0, 1> L10;  // 4 x 2048, cc2
typedef Tile<float, KIND_LDS, 1, 8, 4, 16, 2, 3, 0, 1> L12; // 4 x 4096, cc2
typedef Tile<float, KIND_LDS, 1, 8, 4, 16, 4, 2, 0, 1> L14; // 4 x 4096, cc4

void register_lds(std::vector<Variant> &r) {
    r.push_back(make_tiled<L0>());
    r.push_back(make_tiled<L1>());
    r.push_back(make_tiled<L2>());
    r.push_back(make_tiled<L3>());
    r.push_back(make_tiled<L4>());
    r.push_back(make_tiled<L5>());
    r.push_back(make_tiled<L6>());
    r.push_back(make_tiled<L7>());
    r.push_back(make_tiled<L8>());
    r.push_back(make_tiled<L10>());
    r.push_back(make_tiled<L12>());
    r.push_back(make_tiled<L14>());
}
}  // namespace dedisp
