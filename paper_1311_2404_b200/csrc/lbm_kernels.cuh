// lbm_kernels.cuh -- sm_100a kernels of the fused stream-and-collide path (Alg. 1).
//
// Store: structure of arrays real[Q][N], x fastest, holding
// the DEVIATION h = f - w (reading A12) of the POST-collision populations (reading A9): the
// step kernel pulls h*_i(x - e_i) (or, behind a SOLID neighbour, its own h*_ibar(x): half-way
// bounce-back, reading A8), collides in registers and writes h*(x) to the other buffer
// with aligned, fully coalesced stores.  Every slot is read once and written once per step.
#pragma once
#include <cuda_runtime.h>
#include "lbm_node.cuh"

namespace lbm {

// Node classes of the uint8 type array (1 B/node of mask traffic, BASELINE.json's byte count).
// Only BOUNDARY nodes read their 4-byte link word.
constexpr uint8_t NODE_BULK = 0, NODE_SOLID = 1, NODE_BOUNDARY = 2;

struct Geom {
    int nx, ny, nz;
    int64_t N;
};

// Element offsets from node n to its periodic neighbours along each axis: m = coordinate - 1,
// p = coordinate + 1 (the lattice is a torus).  Compare-and-select, never '%'.
struct Nbr {
    int xm, xp, ym, yp, zm, zp;
};

__device__ __forceinline__ Nbr neighbours(const Geom &g, int x, int y, int z) {
    Nbr o;
    const int sy = g.nx, sz = g.nx * g.ny;
    o.xm = (x == 0) ? (g.nx - 1) : -1;
    o.xp = (x == g.nx - 1) ? -(g.nx - 1) : 1;
    o.ym = (y == 0) ? (g.ny - 1) * sy : -sy;
    o.yp = (y == g.ny - 1) ? -(g.ny - 1) * sy : sy;
    o.zm = (z == 0) ? (g.nz - 1) * sz : -sz;
    o.zp = (z == g.nz - 1) ? -(g.nz - 1) * sz : sz;
    return o;
}

// Offset of node x + s*e_i relative to x, s = +1 or -1 (compile-time direction table).
template <class L> __device__ __forceinline__ int shift(int i, int s, const Nbr &o) {
    int d = 0;
    const int ex = s * L::ex(i), ey = s * L::ey(i), ez = s * L::ez(i);
    if (ex == 1) d += o.xp; else if (ex == -1) d += o.xm;
    if (ey == 1) d += o.yp; else if (ey == -1) d += o.ym;
    if (ez == 1) d += o.zp; else if (ez == -1) d += o.zm;
    return d;
}

// THE gather rule (reading A8): slot (i' * N + x') of the post-collision store that supplies
// f_i(x, t+1).  Used by the step kernels, the read-out kernels and lbm_get_stream_map alike.
template <class L>
__device__ __forceinline__ int64_t source_slot(int i, int n, int64_t N, const Nbr &o, uint32_t link) {
    return ((link >> i) & 1u) ? (int64_t)L::opp(i) * N + n
                              : (int64_t)i * N + (n + shift<L>(i, -1, o));
}

template <class L, typename T>
__device__ __forceinline__ void gather(const T *__restrict__ src, int n, int64_t N, const Nbr &o,
                                       uint32_t link, T (&h)[L::Q]) {
#pragma unroll
    for (int i = 0; i < L::Q; i++) h[i] = __ldg(src + source_slot<L>(i, n, N, o, link));
}

// Thread -> node: 1-D blocks along x, grid (ceil(nx/BX), ny, nz).
__device__ __forceinline__ bool thread_node(const Geom &g, int &x, int &y, int &z, int &n) {
    x = blockIdx.x * blockDim.x + threadIdx.x;
    y = blockIdx.y;
    z = blockIdx.z;
    n = (z * g.ny + y) * g.nx + x;
    return x < g.nx;
}

// ---- link encoding from the node-type mask (lbm_set_geometry) -------------------------------
template <class L>
__global__ void build_links_kernel(Geom g, const uint8_t *__restrict__ mask, uint8_t *__restrict__ type,
                                   uint32_t *__restrict__ link) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    if (mask[n]) { type[n] = NODE_SOLID; link[n] = LINK_SELF_SOLID; return; }
    const Nbr o = neighbours(g, x, y, z);
    uint32_t w = 0;
#pragma unroll
    for (int i = 1; i < L::Q; i++)
        if (mask[n + shift<L>(i, -1, o)]) w |= 1u << i;
    link[n] = w;
    type[n] = w ? NODE_BOUNDARY : NODE_BULK;
}

__global__ void get_geometry_kernel(Geom g, const uint8_t *__restrict__ type, uint8_t *__restrict__ mask) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    mask[n] = type[n] == NODE_SOLID ? 1 : 0;
}

template <class L>
__global__ void stream_map_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                                  int64_t *__restrict__ map) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    const Nbr o = neighbours(g, x, y, z);
    const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
#pragma unroll
    for (int i = 0; i < L::Q; i++)
        map[(int64_t)i * g.N + n] = (t == NODE_SOLID) ? int64_t(-1) : source_slot<L>(i, n, g.N, o, w);
}

// ---- the fused step: pull-stream + moments + equilibrium + collision (+ Guo) + store ---------
// Rows a1-a8 of DESIGN.md.  One node per thread; Q independent loads are issued before first
// use (bytes in flight), stores are aligned and streaming (each slot is touched once per step).
template <class L, typename T, bool MRT, bool FORCE>
__global__ void __launch_bounds__(256)
step_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
            const T *__restrict__ src, T *__restrict__ dst, Relax<T> rp) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t == NODE_SOLID) return;
    const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    T h[L::Q];
    gather<L, T>(src, n, g.N, o, w, h);
    update_node<L, T, MRT, FORCE>(h, rp);
#pragma unroll
    for (int i = 0; i < L::Q; i++) __stcs(dst + (int64_t)i * g.N + n, h[i]);
}

// ---- canonical <-> internal conversions (off the hot loop; reading A9) ----------------------
// canonical f_i(x,t) -> store: S[source_slot(i,x)] = f_i(x) - w_i (inverse of the gather; the
// gather is a permutation of FLUID slots, so every FLUID slot is written exactly once).
template <class L, typename T>
__global__ void set_distributions_kernel(Geom g, const uint8_t *__restrict__ type,
                                         const uint32_t *__restrict__ link, const T *__restrict__ f,
                                         T *__restrict__ store) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t == NODE_SOLID) return;
    const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
#pragma unroll
    for (int i = 0; i < L::Q; i++)
        store[source_slot<L>(i, n, g.N, o, w)] = f[(int64_t)i * g.N + n] - L::template w<T>(i);
}

// f_i(x,0) = f_i^eq(rho0, u0), eq. (3) (reading A15), scattered like above.
template <class L, typename T>
__global__ void init_equilibrium_kernel(Geom g, const uint8_t *__restrict__ type,
                                        const uint32_t *__restrict__ link, const T *__restrict__ rho0,
                                        const T *__restrict__ u0, T *__restrict__ store) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t == NODE_SOLID) return;
    const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    const T rho = rho0[n];
    T v[3] = {T(0), T(0), T(0)};
#pragma unroll
    for (int a = 0; a < L::D; a++) v[a] = u0[(int64_t)a * g.N + n];
    T heq[L::Q];
    equilibrium_dev<L, T>(rho, rho - T(1), v, heq);
#pragma unroll
    for (int i = 0; i < L::Q; i++) store[source_slot<L>(i, n, g.N, o, w)] = heq[i];
}

template <class L, typename T>
__global__ void get_distributions_kernel(Geom g, const uint8_t *__restrict__ type,
                                         const uint32_t *__restrict__ link, const T *__restrict__ store,
                                         T *__restrict__ f) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t == NODE_SOLID) {
#pragma unroll
        for (int i = 0; i < L::Q; i++) f[(int64_t)i * g.N + n] = T(0);
        return;
    }
    const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    T h[L::Q];
    gather<L, T>(store, n, g.N, o, w, h);
#pragma unroll
    for (int i = 0; i < L::Q; i++) f[(int64_t)i * g.N + n] = h[i] + L::template w<T>(i);
}

// rho = sum f, v = (j + F/2)/rho (eq. 1, eq. 16).  half_g = g/2 (0 for SC2).
template <class L, typename T>
__global__ void macro_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                             const T *__restrict__ store, T *__restrict__ rho_out, T *__restrict__ u_out,
                             T hgx, T hgy, T hgz) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    T rho = T(0), v[3] = {T(0), T(0), T(0)};
    if (t != NODE_SOLID) {
        const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
        const Nbr o = neighbours(g, x, y, z);
        T h[L::Q], drho, j[3];
        gather<L, T>(store, n, g.N, o, w, h);
        moments<L, T>(h, drho, j);
        rho = T(1) + drho;
        const T hg[3] = {hgx, hgy, hgz};
#pragma unroll
        for (int a = 0; a < 3; a++) v[a] = (j[a] + rho * hg[a]) / rho;
    }
    if (rho_out) rho_out[n] = rho;
    if (u_out) {
#pragma unroll
        for (int a = 0; a < L::D; a++) u_out[(int64_t)a * g.N + n] = v[a];
    }
}

// ---- Shan-Chen two-component coupling (eq. 10; two passes) ---------------------
// The pseudopotential is kept as psi(rho) - psi(1): sum_i w_i e_i = 0, so the constant drops out
// of eq. (10) while fp32 keeps ~3 more digits of the density contrast (reading A12).
// PSI = 0: psi = rho  ->  rho - 1;  PSI = 1: psi = 1 - exp(-rho)  ->  -exp(-1) expm1(-(rho - 1)).
template <typename T, int PSI> __device__ __forceinline__ T psi_dev(T drho) {
    if constexpr (PSI == 0) return drho;
    else return T(-0.36787944117144232160) * expm1(-drho);
}
template <typename T, int PSI> __device__ __forceinline__ T psi_one() {
    return PSI == 0 ? T(1) : T(0.63212055882855767840);
}

// Pass 1 (row a9): psi fields of both components from the time-t state.  SOLID: psi = 0 (A14).
template <class L, typename T, int PSI>
__global__ void __launch_bounds__(256)
sc_fields_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                 const T *__restrict__ srcA, const T *__restrict__ srcB, T *__restrict__ psiA,
                 T *__restrict__ psiB) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t == NODE_SOLID) { psiA[n] = -psi_one<T, PSI>(); psiB[n] = -psi_one<T, PSI>(); return; }
    const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    T sA = T(0), sB = T(0);
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        const int64_t s = source_slot<L>(i, n, g.N, o, w);
        sA += __ldg(srcA + s);
        sB += __ldg(srcB + s);
    }
    psiA[n] = psi_dev<T, PSI>(sA);
    psiB[n] = psi_dev<T, PSI>(sB);
}

// sum_i w_i psi(x + e_i) e_i over the neighbour field (18 L1/L2-served reads), in units of 1/36.
template <class L, typename T>
__device__ __forceinline__ void psi_gradient(const T *__restrict__ psi, int n, const Nbr &o, T (&S)[3]) {
    T ax[3] = {T(0), T(0), T(0)}, dg[3] = {T(0), T(0), T(0)};
#pragma unroll
    for (int i = 1; i < L::Q; i++) {
        const T p = __ldg(psi + (n + shift<L>(i, +1, o)));
        const bool axis = (L::ex(i) != 0) + (L::ey(i) != 0) + (L::ez(i) != 0) == 1;
        T(&acc)[3] = axis ? ax : dg;
        if (L::ex(i) == 1) acc[0] += p; else if (L::ex(i) == -1) acc[0] -= p;
        if (L::ey(i) == 1) acc[1] += p; else if (L::ey(i) == -1) acc[1] -= p;
        if (L::ez(i) == 1) acc[2] += p; else if (L::ez(i) == -1) acc[2] -= p;
    }
    // axis weight / diagonal weight = 4 (D2Q9: 1/9 vs 1/36) or 2 (D3Q19: 1/18 vs 1/36)
    const T ratio = L::template w<T>(1) / L::template w<T>(L::Q - 1), wd = L::template w<T>(L::Q - 1);
#pragma unroll
    for (int a = 0; a < 3; a++) S[a] = wd * (ratio * ax[a] + dg[a]);
}

// Pass 2 (rows a10-a11): both components in one kernel: gather, moments, common velocity u'
// (P:188), forces (eq. 10, sign A11) + body force, v_s = u' + F_s / (2 rho_s), LBGK + Guo (A13).
template <class L, typename T, int PSI>
__global__ void __launch_bounds__(256)
sc_step_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
               const T *__restrict__ srcA, const T *__restrict__ srcB, T *__restrict__ dstA,
               T *__restrict__ dstB, const T *__restrict__ psiA, const T *__restrict__ psiB,
               Relax<T> rpA, Relax<T> rpB, T G) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t == NODE_SOLID) return;
    const uint32_t w = (t == NODE_BOUNDARY) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    T hA[L::Q], hB[L::Q];
    gather<L, T>(srcA, n, g.N, o, w, hA);
    gather<L, T>(srcB, n, g.N, o, w, hB);
    T SA[3], SB[3];
    psi_gradient<L, T>(psiA, n, o, SA);
    psi_gradient<L, T>(psiB, n, o, SB);
    T dA, dB, jA[3], jB[3];
    moments<L, T>(hA, dA, jA);
    moments<L, T>(hB, dB, jB);
    const T rA = T(1) + dA, rB = T(1) + dB;
    const T pA = psi_dev<T, PSI>(dA) + psi_one<T, PSI>(), pB = psi_dev<T, PSI>(dB) + psi_one<T, PSI>();
    const T inv_den = T(1) / (rA * rpA.inv_tau + rB * rpB.inv_tau);
    const T irA = T(0.5) / rA, irB = T(0.5) / rB;
    T vA[3], vB[3], FA[3], FB[3];
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const T up = (jA[a] * rpA.inv_tau + jB[a] * rpB.inv_tau) * inv_den;
        FA[a] = -G * pA * SB[a] + rA * rpA.g[a];
        FB[a] = -G * pB * SA[a] + rB * rpB.g[a];
        vA[a] = up + FA[a] * irA;
        vB[a] = up + FB[a] * irB;
    }
    collide<L, T, false, true>(hA, rA, dA, vA, FA, rpA);
#pragma unroll
    for (int i = 0; i < L::Q; i++) __stcs(dstA + (int64_t)i * g.N + n, hA[i]);
    collide<L, T, false, true>(hB, rB, dB, vB, FB, rpB);
#pragma unroll
    for (int i = 0; i < L::Q; i++) __stcs(dstB + (int64_t)i * g.N + n, hB[i]);
}

}  // namespace lbm
