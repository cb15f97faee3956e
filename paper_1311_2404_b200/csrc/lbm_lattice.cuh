// lbm_lattice.cuh -- velocity sets, weights and opposite-direction tables as compile-time
// constants (Table 1; ordering = DESIGN.md reading A2).  Product code: shares nothing
// with oracle/.
#pragma once
#include <stdint.h>

#if defined(__CUDACC__)
#define LBM_HD __host__ __device__ __forceinline__
#else
#define LBM_HD inline
#endif

namespace lbm {

struct D2Q9 {
    static constexpr int Q = 9, D = 2, id = 0;
    // 0 rest; 1 +x 2 +y 3 -x 4 -y; 5 (+,+) 6 (-,+) 7 (-,-) 8 (+,-)
    LBM_HD static constexpr int ex(int i) { constexpr int t[9] = {0, 1, 0, -1, 0, 1, -1, -1, 1}; return t[i]; }
    LBM_HD static constexpr int ey(int i) { constexpr int t[9] = {0, 0, 1, 0, -1, 1, 1, -1, -1}; return t[i]; }
    LBM_HD static constexpr int ez(int) { return 0; }
    LBM_HD static constexpr int opp(int i) { constexpr int t[9] = {0, 3, 4, 1, 2, 7, 8, 5, 6}; return t[i]; }
    // weights by link length 0, 1, sqrt 2: 4/9, 1/9, 1/36
    template <typename T> LBM_HD static constexpr T w(int i) {
        return i == 0 ? T(4) / T(9) : (i < 5 ? T(1) / T(9) : T(1) / T(36));
    }
    LBM_HD static constexpr int w36(int i) { return i == 0 ? 16 : (i < 5 ? 4 : 1); }  // 36 w_i
};

struct D3Q19 {
    static constexpr int Q = 19, D = 3, id = 1;
    // 0 rest; 1 +x 2 -x 3 +y 4 -y 5 +z 6 -z; 7..10 xy diagonals; 11..14 xz; 15..18 yz
    LBM_HD static constexpr int ex(int i) {
        constexpr int t[19] = {0, 1, -1, 0, 0, 0, 0, 1, -1, 1, -1, 1, -1, 1, -1, 0, 0, 0, 0};
        return t[i];
    }
    LBM_HD static constexpr int ey(int i) {
        constexpr int t[19] = {0, 0, 0, 1, -1, 0, 0, 1, 1, -1, -1, 0, 0, 0, 0, 1, -1, 1, -1};
        return t[i];
    }
    LBM_HD static constexpr int ez(int i) {
        constexpr int t[19] = {0, 0, 0, 0, 0, 1, -1, 0, 0, 0, 0, 1, 1, -1, -1, 1, 1, -1, -1};
        return t[i];
    }
    LBM_HD static constexpr int opp(int i) {
        constexpr int t[19] = {0, 2, 1, 4, 3, 6, 5, 10, 9, 8, 7, 14, 13, 12, 11, 18, 17, 16, 15};
        return t[i];
    }
    // weights by link length 0, 1, sqrt 2: 1/3, 1/18, 1/36
    template <typename T> LBM_HD static constexpr T w(int i) {
        return i == 0 ? T(1) / T(3) : (i < 7 ? T(1) / T(18) : T(1) / T(36));
    }
    LBM_HD static constexpr int w36(int i) { return i == 0 ? 12 : (i < 7 ? 2 : 1); }  // 36 w_i
};

// Bit 31 of a node's link word marks the node itself SOLID; bit i (< Q) marks the pull source
// x - e_i SOLID, i.e. population i arrives by half-way bounce-back (reading A8).
constexpr uint32_t LINK_SELF_SOLID = 0x80000000u;
// Bits 30 / 29 repeat the node's WALL_FULLWAY / VELOCITY type, so that the kernel for obstacle-rich
// geometries (step_rows_kernel) needs the link word only, not the type byte as well.
constexpr uint32_t LINK_FULLWAY = 0x40000000u, LINK_VELOCITY = 0x20000000u;
constexpr uint32_t LINK_DIRECTIONS = 0x000ffffeu;  // bits 1 .. 19: "some pull source is SOLID"

}  // namespace lbm
