// variants_u8.cu -- uint8 input, uint32 accumulation/output (BASELINE.json config 4; exact).
#include "variants_common.cuh"

namespace dedisp {
typedef Tile<uint8_t, KIND_LDS, 4, 2, 4, 4, 16, 3, 0, 2> U0;  // 16 x 256
typedef Tile<uint8_t, KIND_LDS, 8, 1, 4, 8, 16, 3, 0, 2> U1;  // 32 x 256
typedef Tile<uint8_t, KIND_LDS, 4, 2, 8, 4, 16, 3, 0, 2> U2;  // 32 x 256
typedef Tile<uint8_t, KIND_LDS, 4, 2, 8, 8, 16, 2, 0, 2> U3;  // 32 x 512
typedef Tile<uint8_t, KIND_LDS, 2, 2, 2, 2, 8, 2, 0, 4> U4;   // 4 x 128

void register_u8(std::vector<Variant> &r) {
    r.push_back(make_tiled<U0>());
    r.push_back(make_tiled<U1>());
    r.push_back(make_tiled<U2>());
    r.push_back(make_tiled<U3>());
    r.push_back(make_tiled<U4>());
}
}  // namespace dedisp
