// lbm_kernels.cuh -- sm_100a kernels of the fused stream-and-collide path (Alg. 1).
//
// Store: structure of arrays real[Q][N], x fastest, holding
// the DEVIATION h = f - w (reading A12) of the POST-collision populations (reading A9).
//   * f_i(x, t+1) is pulled from slot (i, x - e_i) with aligned vector loads for every node;
//     BOUNDARY nodes (>= 1 SOLID pull source) then replace each reflected population by their own
//     h*_ibar(x) from slot (ibar, x) (half-way bounce-back, reading A8).  Only packs that
//     contain a BOUNDARY node execute that fix-up.
//   * a node writes its post-collision h*_i(x) to (i, x) of the other buffer with aligned vector
//     stores.  Slots of SOLID nodes are never read (every pull from them is reflected), so packs
//     that mix FLUID and SOLID nodes still store whole vectors.  Every FLUID slot is read once and
//     written once per step: DRAM traffic is the algorithmic 2 Q sizeof(real) + mask bytes.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <type_traits>
#include "lbm_node.cuh"

namespace lbm {

// Node classes of the uint8 type array (1 B/node of mask traffic, BASELINE.json's byte count),
// as bit flags: SOLID (dry, reflects by half-way bounce-back), LINKS (>= 1 SOLID pull source: the
// node reads its 4-byte link word), FULLWAY (dry full-way bounce-back wall node, A20),
// VELOCITY (equilibrium-velocity node, A21).  0 = BULK fluid.
constexpr uint8_t NODE_BULK = 0, NODE_SOLID = 1, NODE_LINKS = 2, NODE_FULLWAY = 4, NODE_VELOCITY = 8;
constexpr uint32_t PACK_SOLID = 0x01010101u, PACK_LINKS = 0x02020202u, PACK_SPECIAL = 0x0C0C0C0Cu;
// lbm_set_geometry mask values (include/lbm.h)
constexpr uint8_t MASK_FLUID = 0, MASK_SOLID = 1, MASK_FULLWAY = 2, MASK_VELOCITY = 3;
__device__ __forceinline__ bool mask_is_solid(uint8_t m) { return m != MASK_FLUID && m != MASK_FULLWAY && m != MASK_VELOCITY; }

struct Geom {
    int nx, ny, nz;
    int64_t N;
    int z0;  // first z-plane this launch covers (blockIdx.z counts from it): 0 except in lbm_step_slabs
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
// y/z part only (multiples of nx: keeps 16-byte alignment of vector accesses)
template <class L> __device__ __forceinline__ int shift_yz(int i, int s, const Nbr &o) {
    int d = 0;
    const int ey = s * L::ey(i), ez = s * L::ez(i);
    if (ey == 1) d += o.yp; else if (ey == -1) d += o.ym;
    if (ez == 1) d += o.zp; else if (ez == -1) d += o.zm;
    return d;
}

// THE streaming rule (reading A8), shared by the step kernels, the conversion kernels and
// lbm_get_stream_map: population i of a node with link word `link` is reflected iff bit i is set;
// then it comes from the node's own slot (ibar, x) instead of (i, x - e_i).
__device__ __forceinline__ bool reflected(uint32_t link, int i) { return (link >> i) & 1u; }

// I = index type of slot numbers i * N + node: uint32_t when Q * N < 2^32 (one IMAD.WIDE per access
// instead of a 64-bit add chain; the step kernels were issue-bound on address arithmetic), else int64_t.
template <class L, typename I>
__device__ __forceinline__ I source_slot(int i, int n, int64_t N, const Nbr &o, uint32_t link) {
    return reflected(link, i) ? I(L::opp(i)) * I(N) + I(n) : I(i) * I(N) + I(n + shift<L>(i, -1, o));
}

// Replace the reflected populations of one BOUNDARY node (after the plain pull).
template <class L, typename T, typename I>
__device__ __forceinline__ void pull_reflected(const T *__restrict__ src, int n, int64_t N, uint32_t link, T (&h)[L::Q]) {
#pragma unroll
    for (int i = 1; i < L::Q; i++)
        if (reflected(link, i)) h[i] = __ldg(src + (I(L::opp(i)) * I(N) + I(n)));
}

// One node, scalar (conversion kernels).
template <class L, typename T>
__device__ __forceinline__ void gather(const T *__restrict__ src, int n, int64_t N, const Nbr &o, uint32_t link, T (&h)[L::Q]) {
#pragma unroll
    for (int i = 0; i < L::Q; i++) h[i] = __ldg(src + source_slot<L, int64_t>(i, n, N, o, link));
}

// Thread -> node for the one-node-per-thread kernels: 1-D blocks along x.
__device__ __forceinline__ bool thread_node(const Geom &g, int &x, int &y, int &z, int &n) {
    x = blockIdx.x * blockDim.x + threadIdx.x;
    y = blockIdx.y;
    z = blockIdx.z + g.z0;
    n = (z * g.ny + y) * g.nx + x;
    return x < g.nx;
}

// ---- link encoding from the node-type mask (lbm_set_geometry) -------------------------------
template <class L>
__global__ void build_links_kernel(Geom g, const uint8_t *__restrict__ mask, uint8_t *__restrict__ type,
                                   uint32_t *__restrict__ link, unsigned *__restrict__ nonbulk_count) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    uint32_t w = LINK_SELF_SOLID;
    uint8_t t = NODE_SOLID;
    const uint8_t m = mask[n];
    if (!mask_is_solid(m)) {
        const Nbr o = neighbours(g, x, y, z);
        w = 0;
#pragma unroll
        for (int i = 1; i < L::Q; i++)
            if (mask_is_solid(mask[n + shift<L>(i, -1, o)])) w |= 1u << i;
        t = (w ? NODE_LINKS : NODE_BULK) | (m == MASK_FULLWAY ? NODE_FULLWAY : 0) | (m == MASK_VELOCITY ? NODE_VELOCITY : 0);
        w |= (m == MASK_FULLWAY ? LINK_FULLWAY : 0u) | (m == MASK_VELOCITY ? LINK_VELOCITY : 0u);
    }
    link[n] = w;
    type[n] = t;
    // warp-aggregated count of nodes that are not BULK (picks the pack width of the step kernels)
    const unsigned active = __activemask(), votes = __ballot_sync(active, t != NODE_BULK);
    if (votes && (threadIdx.x & 31) == __ffs(active) - 1) atomicAdd(nonbulk_count, __popc(votes));
}

static __global__ void get_geometry_kernel(Geom g, const uint8_t *__restrict__ type, uint8_t *__restrict__ mask) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    mask[n] = (t & NODE_SOLID) ? MASK_SOLID : (t & NODE_FULLWAY) ? MASK_FULLWAY : (t & NODE_VELOCITY) ? MASK_VELOCITY : MASK_FLUID;
}

template <class L>
__global__ void stream_map_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                                  int64_t *__restrict__ map) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    const Nbr o = neighbours(g, x, y, z);
    const uint32_t w = (t & NODE_LINKS) ? link[n] : 0u;
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        map[(int64_t)i * g.N + n] = (t & NODE_SOLID) ? int64_t(-1) : source_slot<L, int64_t>(i, n, g.N, o, w);
    }
}

// ---- V consecutive x-nodes per thread, 16-byte (or 8-byte) global accesses -------------------
template <typename T, int V> struct Pack;
template <typename T> struct Pack<T, 1> {
    static __device__ __forceinline__ void ld(const T *p, T (&a)[1]) { a[0] = __ldg(p); }
    static __device__ __forceinline__ void st(T *p, const T (&a)[1]) { __stcs(p, a[0]); }
    static __device__ __forceinline__ void stp(T *p, const T (&a)[1]) { *p = a[0]; }
    static __device__ __forceinline__ void ldp(const T *p, T (&a)[1]) { a[0] = *p; }
};
template <> struct Pack<float, 2> {
    static __device__ __forceinline__ void ld(const float *p, float (&a)[2]) {
        const float2 v = __ldg(reinterpret_cast<const float2 *>(p)); a[0] = v.x; a[1] = v.y;
    }
    static __device__ __forceinline__ void st(float *p, const float (&a)[2]) {
        __stcs(reinterpret_cast<float2 *>(p), make_float2(a[0], a[1]));
    }
    static __device__ __forceinline__ void ldp(const float *p, float (&a)[2]) {
        const float2 v = *reinterpret_cast<const float2 *>(p); a[0] = v.x; a[1] = v.y;
    }
    static __device__ __forceinline__ void stp(float *p, const float (&a)[2]) {
        *reinterpret_cast<float2 *>(p) = make_float2(a[0], a[1]);
    }
};
template <> struct Pack<float, 4> {
    static __device__ __forceinline__ void ld(const float *p, float (&a)[4]) {
        const float4 v = __ldg(reinterpret_cast<const float4 *>(p)); a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w;
    }
    static __device__ __forceinline__ void st(float *p, const float (&a)[4]) {
        __stcs(reinterpret_cast<float4 *>(p), make_float4(a[0], a[1], a[2], a[3]));
    }
    static __device__ __forceinline__ void ldp(const float *p, float (&a)[4]) {
        const float4 v = *reinterpret_cast<const float4 *>(p); a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w;
    }
    static __device__ __forceinline__ void stp(float *p, const float (&a)[4]) {
        *reinterpret_cast<float4 *>(p) = make_float4(a[0], a[1], a[2], a[3]);
    }
};
template <> struct Pack<double, 2> {
    static __device__ __forceinline__ void ld(const double *p, double (&a)[2]) {
        const double2 v = __ldg(reinterpret_cast<const double2 *>(p)); a[0] = v.x; a[1] = v.y;
    }
    static __device__ __forceinline__ void st(double *p, const double (&a)[2]) {
        __stcs(reinterpret_cast<double2 *>(p), make_double2(a[0], a[1]));
    }
    static __device__ __forceinline__ void ldp(const double *p, double (&a)[2]) {
        const double2 v = *reinterpret_cast<const double2 *>(p); a[0] = v.x; a[1] = v.y;
    }
    static __device__ __forceinline__ void stp(double *p, const double (&a)[2]) {
        *reinterpret_cast<double2 *>(p) = make_double2(a[0], a[1]);
    }
};

// A thread's V nodes: x0 .. x0+V-1 of row (y, z); nx % V == 0 so a pack never straddles a row.
struct Span {
    int x0, y, z;
    int row;     // node index of (0, y, z)
    int xm, xp;  // x-coordinate left of x0 and right of x0+V-1 on the torus
    Nbr o;       // o.xm / o.xp unused here (per-node x offsets differ inside the pack)
};

// Threads are numbered along the packs of a z-plane, x fastest, rows following one another without padding:
// a block covers blockDim.x consecutive packs wherever a row ends, so no lane idles on lattices whose
// nx / V is not a multiple of the block width (320^3 at V = 4: 80 packs per row under 64-wide blocks left
// 37 % of the lanes of every second block empty; 38.8 -> 43 GLUPS).
template <int V> __device__ __forceinline__ bool thread_span(const Geom &g, Span &s) {
    const unsigned nxv = (unsigned)g.nx / V, p = blockIdx.x * blockDim.x + threadIdx.x;
    s.y = (int)(p / nxv);
    s.x0 = (int)(p - (unsigned)s.y * nxv) * V;
    s.z = blockIdx.z + g.z0;
    if (s.y >= g.ny) return false;
    s.row = (s.z * g.ny + s.y) * g.nx;
    s.xm = (s.x0 == 0) ? g.nx - 1 : s.x0 - 1;
    s.xp = (s.x0 + V == g.nx) ? 0 : s.x0 + V;
    s.o = neighbours(g, 1, s.y, s.z);
    return true;
}

// Pull for V nodes (row a2): e_x = 0 planes with one aligned vector load; e_x = +-1 planes with
// the aligned vector of the source row plus ONE scalar for the element that falls outside the
// pack (an L1 hit: the neighbouring thread's vector load brings the same sector).
template <class L, typename T, int V, typename I>
__device__ __forceinline__ void gather_span(const T *__restrict__ src, int64_t N, const Span &s, T (&h)[V][L::Q]) {
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        const int r = s.row + shift_yz<L>(i, -1, s.o);  // node index of x = 0 in the source row
        const I plane = I(i) * I(N);
        if (L::ex(i) == 0) {
            T a[V];
            Pack<T, V>::ld(src + (plane + I(r + s.x0)), a);
#pragma unroll
            for (int k = 0; k < V; k++) h[k][i] = a[k];
        } else if (L::ex(i) == 1) {  // source x - 1
            h[0][i] = __ldg(src + (plane + I(r + s.xm)));
            if (V > 1) {
                T a[V];
                Pack<T, V>::ld(src + (plane + I(r + s.x0)), a);
#pragma unroll
                for (int k = 1; k < V; k++) h[k][i] = a[k - 1];
            }
        } else {  // source x + 1
            h[V - 1][i] = __ldg(src + (plane + I(r + s.xp)));
            if (V > 1) {
                T a[V];
                Pack<T, V>::ld(src + (plane + I(r + s.x0)), a);
#pragma unroll
                for (int k = 0; k < V - 1; k++) h[k][i] = a[k + 1];
            }
        }
    }
}

// Node types of the pack as one word (byte k = node k).
// type == nullptr: the geometry has BULK nodes only (all-FLUID torus, e.g. c1 and c5): no load, and the
// thread does not wait one memory round trip before it issues its pull.
template <int V> __device__ __forceinline__ uint32_t load_types(const uint8_t *__restrict__ type, int n0) {
    if (!type) return 0u;
    if (V == 4) return __ldg(reinterpret_cast<const uint32_t *>(type + n0));
    if (V == 2) return __ldg(reinterpret_cast<const uint16_t *>(type + n0));
    return __ldg(type + n0);
}
template <int V> __device__ __forceinline__ bool all_solid(uint32_t t) {
    return t == (V == 4 ? 0x01010101u : V == 2 ? 0x0101u : 0x01u);
}

// Fix-up of the pack's BOUNDARY nodes (row a2, reflected links).
template <class L, typename T, int V, typename I>
__device__ __forceinline__ void pull_reflected_span(const T *__restrict__ src, int64_t N, int n0, uint32_t types,
                                                    const uint32_t *__restrict__ link, T (&h)[V][L::Q]) {
    if (types & PACK_LINKS) {
#pragma unroll
        for (int k = 0; k < V; k++)
            if (((types >> (8 * k)) & 0xffu) & NODE_LINKS)
                pull_reflected<L, T, I>(src, n0 + k, N, __ldg(link + n0 + k), h[k]);
    }
}

// Store for V nodes (row a8): aligned vector, streaming.
template <class L, typename T, int V, typename I>
__device__ __forceinline__ void store_span(T *__restrict__ dst, int64_t N, int n0, const T (&h)[V][L::Q]) {
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        T a[V];
#pragma unroll
        for (int k = 0; k < V; k++) a[k] = h[k][i];
        Pack<T, V>::st(dst + (I(i) * I(N) + I(n0)), a);
    }
}

// Collision by node type (t = the node's type byte).
template <class L, typename T, int MODEL, int FORCE>
__device__ __forceinline__ void update_typed(T (&h)[L::Q], uint32_t t, const Relax<T> &rp) {
    if (t & NODE_FULLWAY) fullway_reverse<L, T>(h);
    else if (t & NODE_VELOCITY) velocity_node<L, T>(h, rp.ubc);
    else update_node<L, T, MODEL, FORCE>(h, rp);
}

// All nodes of a pack; packs without FULLWAY / VELOCITY nodes take the branch-free path.
template <class L, typename T, int V, int MODEL, int FORCE>
__device__ __forceinline__ void update_span(T (&h)[V][L::Q], uint32_t types, const Relax<T> &rp) {
    if ((types & PACK_SPECIAL) == 0) {
#pragma unroll
        for (int k = 0; k < V; k++) update_node<L, T, MODEL, FORCE>(h[k], rp);
    } else {
#pragma unroll
        for (int k = 0; k < V; k++) update_typed<L, T, MODEL, FORCE>(h[k], (types >> (8 * k)) & 0xffu, rp);
    }
}

// ---- the fused step: pull-stream + moments + equilibrium + collision (+ Guo) + store ---------
// Rows a1-a8 of DESIGN.md.  All loads of the pack are issued before first use (bytes in flight).
template <class L, typename T, int V, typename I, int MODEL, int FORCE>
__global__ void __launch_bounds__(256)
step_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
            const T *__restrict__ src, T *__restrict__ dst, Relax<T> rp) {
    Span s;
    if (!thread_span<V>(g, s)) return;
    const int n0 = s.row + s.x0;
    const uint32_t types = load_types<V>(type, n0);
    if (all_solid<V>(types)) return;
    T h[V][L::Q];
    gather_span<L, T, V, I>(src, g.N, s, h);
    pull_reflected_span<L, T, V, I>(src, g.N, n0, types, link, h);
    update_span<L, T, V, MODEL, FORCE>(h, types, rp);
    store_span<L, T, V, I>(dst, g.N, s.row + s.x0, h);
}

// ---- the fused step for obstacle-rich geometries (c3: 57 % of the fluid nodes touch a SOLID) ---
// step_kernel re-pulls reflected links after the link word has arrived: a second, dependent memory
// round trip per thread, which at 80 registers / 24 warps per SM left it latency-bound (r01e: 68 % of
// the DRAM peak, 74 % of the stall samples on long_scoreboard).  Here a thread walks `rows`
// consecutive y-rows of one x-span and fetches the link words of row y+1 while row y is in flight,
// so that when a row starts its link words are already in registers and EVERY population load --
// pulled from (i, x - e_i) or, for a reflected link, from the node's own (ibar, x) -- is issued in
// one batch with the address selected per lane: one round trip, no fix-up pass.  Loads are scalar
// per node (a lane's source depends on its own link bit), the arithmetic and the aligned vector
// stores stay V nodes wide.  Only the link array is read (it repeats the node types, lbm_lattice.cuh).
template <class L, int V> __device__ __forceinline__ uint32_t types_of_links(const uint32_t (&w)[V]) {
    uint32_t types = 0;
#pragma unroll
    for (int k = 0; k < V; k++) {
        const uint32_t t = (w[k] >> 31) | ((w[k] & LINK_DIRECTIONS) ? NODE_LINKS : 0u) |
                           ((w[k] & LINK_FULLWAY) ? NODE_FULLWAY : 0u) | ((w[k] & LINK_VELOCITY) ? NODE_VELOCITY : 0u);
        types |= t << (8 * k);
    }
    return types;
}

template <class L, typename T, int V, typename I>
__device__ __forceinline__ void gather_selected_span(const T *__restrict__ src, int64_t N, const Span &s,
                                                     const uint32_t (&w)[V], T (&h)[V][L::Q]) {
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        const int r = s.row + shift_yz<L>(i, -1, s.o);
        const I plane = I(i) * I(N), own = I(L::opp(i)) * I(N) + I(s.row + s.x0);
#pragma unroll
        for (int k = 0; k < V; k++) {
            const int xs = L::ex(i) == 0 ? s.x0 + k
                         : L::ex(i) == 1 ? (k == 0 ? s.xm : s.x0 + k - 1)
                                         : (k == V - 1 ? s.xp : s.x0 + k + 1);
            const I idx = (i > 0 && reflected(w[k], i)) ? own + I(k) : plane + I(r + xs);
            h[k][i] = __ldg(src + idx);
        }
    }
}

template <int V> __device__ __forceinline__ void load_links(const uint32_t *__restrict__ link, int n0, uint32_t (&w)[V]) {
    if (V == 4) { const uint4 v = __ldg(reinterpret_cast<const uint4 *>(link + n0)); w[0] = v.x; w[1 % V] = v.y; w[2 % V] = v.z; w[V - 1] = v.w; }
    else if (V == 2) { const uint2 v = __ldg(reinterpret_cast<const uint2 *>(link + n0)); w[0] = v.x; w[V - 1] = v.y; }
    else w[0] = __ldg(link + n0);
}

// 64-thread blocks (128 allowed); fp32: 80 registers (24 warps per SM), fp64: 168 registers, by measurement
// on c3 (fp32 at 96 registers / 20 warps: the same; at 64 registers / 32 warps: -10 %, spills).
template <class L, typename T, int V, typename I, int MODEL, int FORCE>
__global__ void __launch_bounds__(128, sizeof(T) == 4 ? 6 : 3)
step_rows_kernel(Geom g, const uint32_t *__restrict__ link, const T *__restrict__ src, T *__restrict__ dst,
                 Relax<T> rp, int rows) {
    Span s;  // threads numbered along (x-pack, y-chunk), x fastest, chunk rows back to back (no idle lanes, see thread_span)
    const unsigned nxv = (unsigned)g.nx / V, p = blockIdx.x * blockDim.x + threadIdx.x, chunk = p / nxv;
    s.x0 = (int)(p - chunk * nxv) * V;
    const int y0 = (int)chunk * rows, y1 = min(y0 + rows, g.ny);
    if (y0 >= g.ny) return;
    s.z = blockIdx.z + g.z0;
    s.xm = (s.x0 == 0) ? g.nx - 1 : s.x0 - 1;
    s.xp = (s.x0 + V == g.nx) ? 0 : s.x0 + V;
    uint32_t wn[V];
    load_links<V>(link, (s.z * g.ny + y0) * g.nx + s.x0, wn);
    for (int y = y0; y < y1; y++) {
        uint32_t w[V];
#pragma unroll
        for (int k = 0; k < V; k++) w[k] = wn[k];
        s.y = y;
        s.row = (s.z * g.ny + y) * g.nx;
        s.o = neighbours(g, 1, y, s.z);
        if (y + 1 < y1) load_links<V>(link, s.row + g.nx + s.x0, wn);  // next row: in flight during this row's pull
        const uint32_t types = types_of_links<L, V>(w);
        if (all_solid<V>(types)) continue;
        T h[V][L::Q];
        gather_selected_span<L, T, V, I>(src, g.N, s, w, h);
        update_span<L, T, V, MODEL, FORCE>(h, types, rp);
        store_span<L, T, V, I>(dst, g.N, s.row + s.x0, h);
    }
}

// The same kernel with the thread's NPT nodes apart instead of adjacent (nx % NPT == 0): one warp width apart where
// whole warps tile a row (lane l of warp w owns x = 32 NPT w + l + 32 k), else thread q of a row owns x = q + k nx / NPT,
// so that consecutive lanes own consecutive nodes.  The per-lane source select forces scalar loads
// either way; adjacent nodes make a warp's 4-byte loads stride 8 bytes (every sector requested twice, half of
// it used: 330 M L1 sector requests for 4.5 GB of populations on c3), nodes part of a row apart make every load and
// store instruction of a warp one contiguous 128-byte line (4 whole sectors; 5 for the e_x = +-1 planes).
template <class L, typename T, int NPT, typename I, int MODEL, int FORCE>
__global__ void __launch_bounds__(128, sizeof(T) == 4 ? 6 : 3)
step_rows_strided_kernel(Geom g, const uint32_t *__restrict__ link, const T *__restrict__ src, T *__restrict__ dst,
                         Relax<T> rp, int rows) {
    const unsigned per_row = (unsigned)g.nx / NPT, p = blockIdx.x * blockDim.x + threadIdx.x, chunk = p / per_row;
    // x of node k = xb + k XS: one warp width apart where whole warps tile the row (3 % faster on c3: a thread's two
    // lines lie side by side), else the row in NPT equal parts
    const unsigned q = p - chunk * per_row;
    const bool tiled = g.nx % (32 * NPT) == 0;
    const int xb = tiled ? (int)(q >> 5) * (32 * NPT) + (int)(q & 31u) : (int)q, XS = tiled ? 32 : (int)per_row;
    const int y0 = (int)chunk * rows, y1 = min(y0 + rows, g.ny);
    if (y0 >= g.ny) return;
    const int z = blockIdx.z + g.z0;
    int xm[NPT], xp[NPT];  // periodic x - 1 / x + 1 of each node
#pragma unroll
    for (int k = 0; k < NPT; k++) {
        const int x = xb + XS * k;
        xm[k] = x == 0 ? g.nx - 1 : x - 1;
        xp[k] = x == g.nx - 1 ? 0 : x + 1;
    }
    uint32_t wn[NPT];
#pragma unroll
    for (int k = 0; k < NPT; k++) wn[k] = __ldg(link + ((z * g.ny + y0) * g.nx + xb + XS * k));
    for (int y = y0; y < y1; y++) {
        uint32_t w[NPT];
#pragma unroll
        for (int k = 0; k < NPT; k++) w[k] = wn[k];
        const int row = (z * g.ny + y) * g.nx;
        const Nbr o = neighbours(g, 1, y, z);
        if (y + 1 < y1) {
#pragma unroll
            for (int k = 0; k < NPT; k++) wn[k] = __ldg(link + (row + g.nx + xb + XS * k));
        }
        const uint32_t types = types_of_links<L, NPT>(w);
        T h[NPT][L::Q];
#pragma unroll
        for (int i = 0; i < L::Q; i++) {
            const int r = row + shift_yz<L>(i, -1, o);
            const I plane = I(i) * I(g.N), own = I(L::opp(i)) * I(g.N) + I(row + xb);
#pragma unroll
            for (int k = 0; k < NPT; k++) {
                const int xs = L::ex(i) == 0 ? xb + XS * k : L::ex(i) == 1 ? xm[k] : xp[k];
                const I idx = (i > 0 && reflected(w[k], i)) ? own + I(XS * k) : plane + I(r + xs);
                h[k][i] = __ldg(src + idx);
            }
        }
        // SOLID nodes run through as well (on whatever their pull returned) and store: a warp's store is then
        // always four whole sectors; nothing ever reads a SOLID node's slots
        update_span<L, T, NPT, MODEL, FORCE>(h, types & ~PACK_SOLID, rp);
#pragma unroll
        for (int i = 0; i < L::Q; i++)
#pragma unroll
            for (int k = 0; k < NPT; k++) __stcs(dst + (I(i) * I(g.N) + I(row + xb + XS * k)), h[k][i]);
    }
}

// ---- z-slab decomposition: ghost-plane exchange ------------------------------------
// A slab context holds its share of the lattice as local planes 1 .. nz-2 plus one ghost plane below
// (0) and above (nz-1).  After a step the ghost planes receive, from the neighbouring slab's boundary
// interior plane, the populations that will stream across the face ("only the mass fractions that
// actually need to be sent"): in the SoA store a population's z-plane is one contiguous run of
// nx*ny values, so the "pack" is a plane copy per crossing direction (5 of 19 for D3Q19).  The same
// kernel moves the psi planes of the Shan-Chen fields (ndir = 1 per field).  src and dst may live on
// different devices with peer access enabled (plain stores over NVLink); tested on one device.
struct PlaneList { int dir[8]; };
template <typename T>
__global__ void slab_copy_planes_kernel(const T *__restrict__ src, T *__restrict__ dst, int64_t Nsrc, int64_t Ndst,
                                        int64_t src_off, int64_t dst_off, int plane_nodes, PlaneList dirs) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= plane_nodes) return;
    const int i = dirs.dir[blockIdx.y];
    dst[(int64_t)i * Ndst + dst_off + j] = src[(int64_t)i * Nsrc + src_off + j];
}

// ---- canonical <-> internal conversions (off the hot loop; reading A9) ----------------------
// canonical f_i(x,t) -> store: S[source_slot(i, x)] = f_i(x) - w_i, the inverse of the pull.  The
// pull is a permutation of FLUID slots (A8), so every FLUID slot is written exactly once.
template <class L, typename T>
__global__ void set_distributions_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                                         const T *__restrict__ f, T *__restrict__ store) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t & NODE_SOLID) return;
    const uint32_t w = (t & NODE_LINKS) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
#pragma unroll
    for (int i = 0; i < L::Q; i++)
        store[source_slot<L, int64_t>(i, n, g.N, o, w)] = f[(int64_t)i * g.N + n] - L::template w<T>(i);
}

// f_i(x,0) = f_i^eq(rho0, u0), eq. (3) (reading A15), scattered like above.
template <class L, typename T>
__global__ void init_equilibrium_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                                        const T *__restrict__ rho0, const T *__restrict__ u0, T *__restrict__ store) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t & NODE_SOLID) return;
    const uint32_t w = (t & NODE_LINKS) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    const T rho = rho0[n];
    T v[3] = {T(0), T(0), T(0)};
#pragma unroll
    for (int a = 0; a < L::D; a++) v[a] = u0[(int64_t)a * g.N + n];
    T heq[L::Q];
    equilibrium_dev<L, T>(rho, rho - T(1), v, heq);
#pragma unroll
    for (int i = 0; i < L::Q; i++) store[source_slot<L, int64_t>(i, n, g.N, o, w)] = heq[i];
}

template <class L, typename T>
__global__ void get_distributions_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                                         const T *__restrict__ store, T *__restrict__ f) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    if (t & NODE_SOLID) {
#pragma unroll
        for (int i = 0; i < L::Q; i++) f[(int64_t)i * g.N + n] = T(0);
        return;
    }
    const uint32_t w = (t & NODE_LINKS) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    T h[L::Q];
    gather<L, T>(store, n, g.N, o, w, h);
#pragma unroll
    for (int i = 0; i < L::Q; i++) f[(int64_t)i * g.N + n] = h[i] + L::template w<T>(i);
}

// rho = sum f, v = (j + F/2)/rho (eq. 1, eq. 16).  hg = g/2 (0 for SC2).
template <class L, typename T>
__global__ void macro_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                             const T *__restrict__ store, T *__restrict__ rho_out, T *__restrict__ u_out,
                             T hgx, T hgy, T hgz) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    T rho = T(0), v[3] = {T(0), T(0), T(0)};
    if (!(t & (NODE_SOLID | NODE_FULLWAY))) {  // dry nodes report rho = 0, u = 0
        const uint32_t w = (t & NODE_LINKS) ? link[n] : 0u;
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

// ---- small lattices: the whole AB store resident in the shared memory of one thread-block cluster ---
// The paper's saturation plot is the launch-bound regime: a 128^2 D2Q9 lattice is 0.6 MB
// per buffer and one step of it takes ~2 us however it is launched.  Here CTA r of a cluster of 8
// (portable) or 16 (non-portable size, D2Q9 only) CTAs keeps slots [Q][S] of nodes [r S, (r+1) S) of
// both buffers in its shared memory, one node per thread; a pull from a node owned by another CTA
// is a distributed-shared-memory load, steps are separated by cluster.sync(), and global memory is
// touched only before the first and after the last step of an lbm_step(n) call.  A node's Q source
// addresses (shared::cluster window, reflected links resolved) never change, so they are computed
// once and kept in registers.  Same arithmetic and streaming rule as step_kernel: bit-identical.
constexpr int RESIDENT_MAX_CTAS = 16;

// SFIX: the CTA's share S equals THREADS (a compile-time constant).  Then the step loop is unrolled by two
// (one body per buffer parity) and every shared-memory address is a register that never changes plus an
// immediate: 9 LD + 9 STS + the collision per D2Q9 node and step, no address arithmetic (the generic-S loop
// spends half of its issue slots on it, and at 1024 nodes per SM the kernel is issue-bound).
template <class L, typename T, int MODEL, int FORCE, int THREADS, bool SFIX>
__global__ void __launch_bounds__(THREADS)
resident_kernel(Geom g, int s_log2_arg, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                const T *src, T *dst, Relax<T> rp, int nsteps) {
    extern __shared__ __align__(16) unsigned char resident_smem[];
    T *buf = reinterpret_cast<T *>(resident_smem);  // [2][Q][S]
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    constexpr int LOG2_THREADS = THREADS == 1024 ? 10 : THREADS == 512 ? 9 : THREADS == 256 ? 8 : 7;
    static_assert((1 << LOG2_THREADS) == THREADS, "THREADS must be 128 .. 1024, a power of two");
    const int s_log2 = SFIX ? LOG2_THREADS : s_log2_arg;
    const int S = 1 << s_log2, mask = S - 1, N = (int)g.N;
    const int base = (int)cluster.block_rank() * S;
    const int tid = threadIdx.x;
    if constexpr (SFIX) {  // S == THREADS: one slot of every plane per thread, all Q loads in flight at once
        T v[L::Q];
#pragma unroll
        for (int i = 0; i < L::Q; i++) v[i] = base + tid < N ? src[(int64_t)i * N + base + tid] : T(0);
#pragma unroll
        for (int i = 0; i < L::Q; i++) buf[i * THREADS + tid] = v[i];
    } else {
        for (int idx = tid; idx < L::Q * S; idx += THREADS) {
            const int i = idx >> s_log2, n = base + (idx & mask);
            buf[idx] = n < N ? src[(int64_t)i * N + n] : T(0);
        }
    }
    // this thread's node: type and the Q source addresses (buffer 0; generic pointers into the cluster's
    // distributed shared memory, reflected links resolved) stay in registers for all steps
    const int n = base + tid;
    uint32_t t = NODE_SOLID;  // threads beyond the lattice or beyond S do nothing
    const T *from[L::Q];
#pragma unroll
    for (int i = 0; i < L::Q; i++) from[i] = buf;
    if (tid < S && n < N) {
        t = type[n];
        const uint32_t w = (t & NODE_LINKS) ? link[n] : 0u;
        const int x = n % g.nx, y = (n / g.nx) % g.ny, z = n / (g.nx * g.ny);
        const Nbr o = neighbours(g, x, y, z);
#pragma unroll
        for (int i = 0; i < L::Q; i++) {
            const bool refl = reflected(w, i);
            const int m = refl ? n : n + shift<L>(i, -1, o);  // source node
            const int plane = refl ? L::opp(i) : i;
            from[i] = cluster.map_shared_rank(buf + plane * S + (m & mask), m >> s_log2);
        }
    }
    T *mine = buf + tid;
    cluster.sync();
    int cur = 0;
    if constexpr (SFIX) {
        constexpr int FLIP = L::Q * THREADS;  // elements between the two buffers
        auto one_step = [&](auto parity) {
            constexpr int c = decltype(parity)::value;
            if (!(t & NODE_SOLID)) {
                T h[L::Q];
#pragma unroll
                for (int i = 0; i < L::Q; i++) h[i] = from[i][c * FLIP];
                update_typed<L, T, MODEL, FORCE>(h, t, rp);
#pragma unroll
                for (int i = 0; i < L::Q; i++) mine[(c ^ 1) * FLIP + i * THREADS] = h[i];
            }
            cluster.sync();  // every CTA has written step t+1 before anyone pulls from it
        };
        int step = 0;
        for (; step + 1 < nsteps; step += 2) {
            one_step(std::integral_constant<int, 0>{});
            one_step(std::integral_constant<int, 1>{});
        }
        if (step < nsteps) { one_step(std::integral_constant<int, 0>{}); cur = 1; }
    } else {
        const int flip = L::Q * S;
        for (int step = 0; step < nsteps; step++) {
            if (!(t & NODE_SOLID)) {
                T h[L::Q];
#pragma unroll
                for (int i = 0; i < L::Q; i++) h[i] = from[i][cur ? flip : 0];
                update_typed<L, T, MODEL, FORCE>(h, t, rp);
                T *B = mine + (cur ^ 1) * flip;
#pragma unroll
                for (int i = 0; i < L::Q; i++) B[i * S] = h[i];
            }
            cluster.sync();
            cur ^= 1;
        }
    }
    for (int idx = tid; idx < L::Q * S; idx += THREADS) {
        const int i = idx >> s_log2, m = base + (idx & mask);
        if (m < N) dst[(int64_t)i * N + m] = buf[cur * L::Q * S + idx];
    }
}

// ---- in-place AA access pattern (row a12; Fig. 4) ---------------------------------
// One buffer.  Before an EVEN step slot (i, x) holds the canonical f_i(x, t) - w_i.  The even step is
// purely local: read (i, x), collide, write h*_i(x) to (ibar, x).  Before an ODD step the canonical
// f_i(x, t) therefore sits in slot (ibar, x - e_i), or for a reflected link in the node's own slot
// (i, x); the odd step reads those, collides, and writes h*_i(x) to the slot its read of ibar came
// from, i.e. (i, x + e_i), or (ibar, x) when x + e_i is SOLID -- which is where the next even step
// expects f(t+2).  Every thread reads and writes exactly the same set of slots.
template <class L, typename I>
__device__ __forceinline__ I aa_slot(int parity, int i, int n, int64_t N, const Nbr &o, uint32_t link) {
    if (parity == 0) return I(i) * I(N) + I(n);
    return reflected(link, i) ? I(i) * I(N) + I(n) : I(L::opp(i)) * I(N) + I(n + shift<L>(i, -1, o));
}

template <class L, typename T, int V, typename I, int MODEL, int FORCE>
__global__ void __launch_bounds__(256)
aa_even_kernel(Geom g, const uint8_t *__restrict__ type, T *f, Relax<T> rp) {
    Span s;
    if (!thread_span<V>(g, s)) return;
    const int n0 = s.row + s.x0;
    const uint32_t types = load_types<V>(type, n0);
    if (all_solid<V>(types)) return;
    T h[V][L::Q];
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        T a[V];
        Pack<T, V>::ldp(f + (I(i) * I(g.N) + I(n0)), a);
#pragma unroll
        for (int k = 0; k < V; k++) h[k][i] = a[k];
    }
    update_span<L, T, V, MODEL, FORCE>(h, types, rp);
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        T a[V];
#pragma unroll
        for (int k = 0; k < V; k++) a[k] = h[k][i];
        Pack<T, V>::stp(f + (I(L::opp(i)) * I(g.N) + I(n0)), a);
    }
}

// ---- odd AA step with V-node packs --------------------------------------------------------------
// Packs whose nodes are all wet with no SOLID pull source ("plain") move whole vectors: the reads are
// the pull of step_kernel from the opposite planes (aligned vector + one scalar for e_x = +-1); the
// writes go to (i, x + e_i), which for e_x = +-1 is the pack's own aligned vector shifted by one node:
// the element that falls on the pack's first (last) column comes from the left (right) neighbour
// thread through shared memory, so that every thread still issues one aligned 16-byte store per plane;
// only the first / last thread of a block row stores its edge elements one by one.  A thread that
// writes on behalf of its neighbour does so after the barrier, i.e. after the neighbour's collision and
// hence after the neighbour has read that slot: the in-place update stays race-free.  Other packs (a SOLID
// node, a reflected link) take the one-node-at-a-time path with link-dependent slots (aa_slot).
template <int V> __device__ __forceinline__ bool pack_plain(uint32_t types) { return (types & (PACK_SOLID | PACK_LINKS)) == 0; }

__device__ __forceinline__ Nbr span_node_neighbours(const Geom &g, const Span &s, int k) {
    Nbr o = s.o;
    const int x = s.x0 + k;
    o.xm = (x == 0) ? (g.nx - 1) : -1;
    o.xp = (x == g.nx - 1) ? -(g.nx - 1) : 1;
    return o;
}

template <int V> __device__ __forceinline__ bool thread_span_all(const Geom &g, Span &s) {
    const unsigned nxv = (unsigned)g.nx / V, p = blockIdx.x * blockDim.x + threadIdx.x;
    s.y = (int)(p / nxv);
    s.x0 = (int)(p - (unsigned)s.y * nxv) * V;
    s.z = blockIdx.z + g.z0;
    const bool valid = s.y < g.ny;
    const int y = valid ? s.y : 0;
    s.row = (s.z * g.ny + y) * g.nx;
    s.xm = (s.x0 == 0) ? g.nx - 1 : s.x0 - 1;
    s.xp = (s.x0 + V == g.nx) ? 0 : s.x0 + V;
    s.o = neighbours(g, 1, y, s.z);
    return valid;
}

// f_i(x, t) before an odd step: slot (ibar, x - e_i), or the node's own (i, x) for a reflected link.
template <class L, typename T, int V, typename I>
__device__ __forceinline__ void aa_gather_odd_span(const T *f, const Geom &g, const Span &s, uint32_t types,
                                                   const uint32_t *__restrict__ link, T (&h)[V][L::Q]) {
    const int64_t N = g.N;
    if (pack_plain<V>(types)) {
#pragma unroll
        for (int i = 0; i < L::Q; i++) {
            const int r = s.row + shift_yz<L>(i, -1, s.o);
            const I plane = I(L::opp(i)) * I(N);
            if (L::ex(i) == 0) {
                T a[V];
                Pack<T, V>::ldp(f + (plane + I(r + s.x0)), a);
#pragma unroll
                for (int k = 0; k < V; k++) h[k][i] = a[k];
            } else if (L::ex(i) == 1) {
                h[0][i] = f[plane + I(r + s.xm)];
                if (V > 1) {
                    T a[V];
                    Pack<T, V>::ldp(f + (plane + I(r + s.x0)), a);
#pragma unroll
                    for (int k = 1; k < V; k++) h[k][i] = a[k - 1];
                }
            } else {
                h[V - 1][i] = f[plane + I(r + s.xp)];
                if (V > 1) {
                    T a[V];
                    Pack<T, V>::ldp(f + (plane + I(r + s.x0)), a);
#pragma unroll
                    for (int k = 0; k < V - 1; k++) h[k][i] = a[k + 1];
                }
            }
        }
    } else {
#pragma unroll
        for (int k = 0; k < V; k++) {
            const uint32_t t = (types >> (8 * k)) & 0xffu;
            const int n = s.row + s.x0 + k;
            const uint32_t w = (t & NODE_LINKS) ? __ldg(link + n) : 0u;
            const Nbr o = span_node_neighbours(g, s, k);
#pragma unroll
            for (int i = 0; i < L::Q; i++) h[k][i] = (t & NODE_SOLID) ? T(0) : f[aa_slot<L, I>(1, i, n, N, o, w)];
        }
    }
}

// h*_i(x) after an odd step: slot (i, x + e_i), or (ibar, x) when x + e_i is SOLID.  Called by EVERY
// thread of the block (`live` = the thread has nodes to write): edge elements travel through shared memory.
constexpr int AA_MAX_BLOCK = 128;  // threads per block of the odd-step AA kernels (lbm_steps.cuh clamps the launch)
template <class L> __device__ __forceinline__ constexpr int edge_slot(int i) {  // rank of link i among those with e_x != 0
    int e = 0;
    for (int j = 1; j < i; j++) e += L::ex(j) != 0;
    return e;
}
template <class L> __device__ __forceinline__ constexpr int edge_count() { return edge_slot<L>(L::Q); }

template <class L, typename T, int V, typename I>
__device__ __forceinline__ void aa_scatter_odd_span(T *f, const Geom &g, const Span &s, uint32_t types, bool live,
                                                    const uint32_t *__restrict__ link, const T (&h)[V][L::Q]) {
    __shared__ T edge[edge_count<L>()][AA_MAX_BLOCK];
    __shared__ uint8_t plain_of[AA_MAX_BLOCK];
    const int64_t N = g.N;
    const int tid = threadIdx.x;  // consecutive threads hold consecutive packs; a row may end inside the block
    const bool plain = live && pack_plain<V>(types);
#pragma unroll
    for (int i = 1; i < L::Q; i++) {  // what the neighbour thread stores on this thread's behalf
        if (L::ex(i) == 1) edge[edge_slot<L>(i)][tid] = h[V - 1][i];
        else if (L::ex(i) == -1) edge[edge_slot<L>(i)][tid] = h[0][i];
    }
    plain_of[tid] = plain;
    __syncthreads();
    const bool has_left = tid > 0 && s.x0 > 0, has_right = tid + 1 < (int)blockDim.x && s.x0 + V < g.nx;  // same row, same block
    const bool left_plain = has_left && plain_of[tid - 1], right_plain = has_right && plain_of[tid + 1];
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        if (!plain) break;
        const int r = s.row + shift_yz<L>(i, +1, s.o);
        const I plane = I(i) * I(N);
        if (L::ex(i) == 0) {
            T a[V];
#pragma unroll
            for (int k = 0; k < V; k++) a[k] = h[k][i];
            Pack<T, V>::stp(f + (plane + I(r + s.x0)), a);
        } else if (L::ex(i) == 1) {  // targets x0 + 1 .. x0 + V
            if (has_left) {
                T a[V];
                a[0] = edge[edge_slot<L>(i)][tid - 1];
#pragma unroll
                for (int k = 1; k < V; k++) a[k] = h[k - 1][i];
                Pack<T, V>::stp(f + (plane + I(r + s.x0)), a);
            } else {
#pragma unroll
                for (int k = 1; k < V; k++) f[plane + I(r + s.x0 + k)] = h[k - 1][i];
            }
            if (!right_plain) f[plane + I(r + s.xp)] = h[V - 1][i];
        } else {  // targets x0 - 1 .. x0 + V - 2
            if (has_right) {
                T a[V];
#pragma unroll
                for (int k = 0; k < V - 1; k++) a[k] = h[k + 1][i];
                a[V - 1] = edge[edge_slot<L>(i)][tid + 1];
                Pack<T, V>::stp(f + (plane + I(r + s.x0)), a);
            } else {
#pragma unroll
                for (int k = 0; k < V - 1; k++) f[plane + I(r + s.x0 + k)] = h[k + 1][i];
            }
            if (!left_plain) f[plane + I(r + s.xm)] = h[0][i];
        }
    }
    if (live && !plain) {
#pragma unroll
        for (int k = 0; k < V; k++) {
            const uint32_t t = (types >> (8 * k)) & 0xffu;
            if (t & NODE_SOLID) continue;
            const int n = s.row + s.x0 + k;
            const uint32_t w = (t & NODE_LINKS) ? __ldg(link + n) : 0u;
            const Nbr o = span_node_neighbours(g, s, k);
#pragma unroll
            for (int i = 0; i < L::Q; i++) f[aa_slot<L, I>(1, L::opp(i), n, N, o, w)] = h[k][i];  // where the read of ibar came from
        }
    }
}

template <class L, typename T, int V, typename I, int MODEL, int FORCE>
__global__ void __launch_bounds__(AA_MAX_BLOCK)
aa_odd_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link, T *f, Relax<T> rp) {
    Span s;
    const bool valid = thread_span_all<V>(g, s);
    const uint32_t types = valid ? load_types<V>(type, s.row + s.x0) : PACK_SOLID;
    const bool live = valid && !all_solid<V>(types);
    T h[V][L::Q];
    if (live) {
        aa_gather_odd_span<L, T, V, I>(f, g, s, types, link, h);
        update_span<L, T, V, MODEL, FORCE>(h, types, rp);
    }
    aa_scatter_odd_span<L, T, V, I>(f, g, s, types, live, link, h);
}

// Odd AA step for obstacle-rich geometries (nx % 64 == 0), in the manner of step_rows_strided_kernel: a thread's
// two nodes lie one warp width apart, the link words come first and every population is then read from the slot
// the streaming rule names -- (ibar, x - e_i), or the node's own (i, x) for a reflected link -- in one batch of
// line-contiguous scalar loads; after the collision h*_i goes to the slot the read of ibar came from.  A node reads
// and writes exactly its own set of slots and all of a thread's loads precede its stores: no hazards.
// SOLID nodes touch nothing (their neighbours' populations live in the slots around them).
template <class L, typename T, int NPT, typename I, int MODEL, int FORCE>
__global__ void __launch_bounds__(128, sizeof(T) == 4 ? 6 : 3)
aa_odd_strided_kernel(Geom g, const uint32_t *__restrict__ link, T *f, Relax<T> rp) {
    const unsigned per_row = (unsigned)g.nx / NPT, p = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = (int)(p / per_row);
    if (y >= g.ny) return;
    const unsigned q = p - (unsigned)y * per_row;
    const bool tiled = g.nx % (32 * NPT) == 0;  // x of node k = xb + k XS, as in step_rows_strided_kernel
    const int xb = tiled ? (int)(q >> 5) * (32 * NPT) + (int)(q & 31u) : (int)q, XS = tiled ? 32 : (int)per_row;
    const int z = blockIdx.z + g.z0, row = (z * g.ny + y) * g.nx;
    const Nbr o = neighbours(g, 1, y, z);
    int xm[NPT], xp[NPT];
    uint32_t w[NPT];
#pragma unroll
    for (int k = 0; k < NPT; k++) {
        const int x = xb + XS * k;
        xm[k] = x == 0 ? g.nx - 1 : x - 1;
        xp[k] = x == g.nx - 1 ? 0 : x + 1;
        w[k] = __ldg(link + (row + x));
    }
    const uint32_t types = types_of_links<L, NPT>(w);
    if (all_solid<NPT>(types)) return;
    T h[NPT][L::Q];
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        const int r = row + shift_yz<L>(i, -1, o);
        const I from = I(L::opp(i)) * I(g.N), own = I(i) * I(g.N) + I(row + xb);
#pragma unroll
        for (int k = 0; k < NPT; k++) {
            const int xs = L::ex(i) == 0 ? xb + XS * k : L::ex(i) == 1 ? xm[k] : xp[k];
            const I idx = (i > 0 && reflected(w[k], i)) ? own + I(XS * k) : from + I(r + xs);
            h[k][i] = (w[k] & LINK_SELF_SOLID) ? T(0) : f[idx];
        }
    }
    update_span<L, T, NPT, MODEL, FORCE>(h, types & ~PACK_SOLID, rp);
#pragma unroll
    for (int i = 0; i < L::Q; i++) {
        const int r = row + shift_yz<L>(i, +1, o);
        const I to = I(i) * I(g.N), own = I(L::opp(i)) * I(g.N) + I(row + xb);
#pragma unroll
        for (int k = 0; k < NPT; k++) {
            const int xs = L::ex(i) == 0 ? xb + XS * k : L::ex(i) == 1 ? xp[k] : xm[k];
            const I idx = (i > 0 && reflected(w[k], L::opp(i))) ? own + I(XS * k) : to + I(r + xs);
            if (!(w[k] & LINK_SELF_SOLID)) f[idx] = h[k][i];
        }
    }
}

// Conversions for the AA store (parity 0: before an even step, 1: before an odd step).
template <class L, typename T, int MODE>  // MODE 0: set from canonical f, 1: get canonical f, 2: init f^eq, 3: macro
__global__ void aa_convert_kernel(Geom g, int parity, const uint8_t *__restrict__ type,
                                  const uint32_t *__restrict__ link, T *store, const T *in0, const T *in1,
                                  T *out0, T *out1, T hgx, T hgy, T hgz) {
    int x, y, z, n;
    if (!thread_node(g, x, y, z, n)) return;
    const uint8_t t = type[n];
    const uint32_t w = (t & NODE_LINKS) ? link[n] : 0u;
    const Nbr o = neighbours(g, x, y, z);
    if (MODE == 0 || MODE == 2) {
        if (t & NODE_SOLID) return;
        T h[L::Q];
        if (MODE == 0) {
#pragma unroll
            for (int i = 0; i < L::Q; i++) h[i] = in0[(int64_t)i * g.N + n] - L::template w<T>(i);
        } else {
            T v[3] = {T(0), T(0), T(0)};
#pragma unroll
            for (int a = 0; a < L::D; a++) v[a] = in1[(int64_t)a * g.N + n];
            equilibrium_dev<L, T>(in0[n], in0[n] - T(1), v, h);
        }
#pragma unroll
        for (int i = 0; i < L::Q; i++) store[aa_slot<L, int64_t>(parity, i, n, g.N, o, w)] = h[i];
    } else {
        T h[L::Q];
#pragma unroll
        for (int i = 0; i < L::Q; i++) h[i] = (t & NODE_SOLID) ? T(0) : store[aa_slot<L, int64_t>(parity, i, n, g.N, o, w)];
        if (MODE == 1) {
#pragma unroll
            for (int i = 0; i < L::Q; i++) out0[(int64_t)i * g.N + n] = (t & NODE_SOLID) ? T(0) : h[i] + L::template w<T>(i);
        } else {
            T rho = T(0), v[3] = {T(0), T(0), T(0)};
            if (!(t & (NODE_SOLID | NODE_FULLWAY))) {
                T drho, j[3];
                moments<L, T>(h, drho, j);
                rho = T(1) + drho;
                const T hg[3] = {hgx, hgy, hgz};
#pragma unroll
                for (int a = 0; a < 3; a++) v[a] = (j[a] + rho * hg[a]) / rho;
            }
            if (out0) out0[n] = rho;
            if (out1) {
#pragma unroll
                for (int a = 0; a < L::D; a++) out1[(int64_t)a * g.N + n] = v[a];
            }
        }
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

template <typename T> struct Pair;
template <> struct Pair<float> { using type = float2; };
template <> struct Pair<double> { using type = double2; };

// Pass 1 (row a9): psi fields of both components from the time-t state.  SOLID: psi = 0 (A14).
template <class L, typename T, int V, typename I, int PSI>
__global__ void __launch_bounds__(256)
sc_fields_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                 const T *__restrict__ srcA, const T *__restrict__ srcB,
                 typename Pair<T>::type *__restrict__ psi) {
    Span s;
    if (!thread_span<V>(g, s)) return;
    const int n0 = s.row + s.x0;
    const uint32_t types = load_types<V>(type, n0);
    T pa[V], pb[V];
    if (all_solid<V>(types)) {
#pragma unroll
        for (int k = 0; k < V; k++) pa[k] = pb[k] = -psi_one<T, PSI>();
    } else {
        T h[V][L::Q];
        gather_span<L, T, V, I>(srcA, g.N, s, h);
        pull_reflected_span<L, T, V, I>(srcA, g.N, n0, types, link, h);
#pragma unroll
        for (int k = 0; k < V; k++) {
            T sum = h[k][0];
#pragma unroll
            for (int i = 1; i < L::Q; i++) sum += h[k][i];
            pa[k] = psi_dev<T, PSI>(sum);
        }
        gather_span<L, T, V, I>(srcB, g.N, s, h);
        pull_reflected_span<L, T, V, I>(srcB, g.N, n0, types, link, h);
#pragma unroll
        for (int k = 0; k < V; k++) {
            T sum = h[k][0];
#pragma unroll
            for (int i = 1; i < L::Q; i++) sum += h[k][i];
            pb[k] = psi_dev<T, PSI>(sum);
            if ((types >> (8 * k)) & (NODE_SOLID | NODE_FULLWAY)) pa[k] = pb[k] = -psi_one<T, PSI>();  // dry: psi = 0 (A14)
        }
    }
    // (psi_A, psi_B) interleaved: pass 2 fetches both with one 8/16-byte load per neighbour.
    // Plain stores: pass 2 re-reads the field right away (L2-resident).
#pragma unroll
    for (int k = 0; k < V; k++) {
        typename Pair<T>::type p;
        p.x = pa[k]; p.y = pb[k];
        psi[n0 + k] = p;
    }
}

// S_A = sum_i w_i psi_A(x + e_i) e_i and S_B likewise, over the interleaved neighbour field
// (18 L1/L2-served reads of both components at once).
template <class L, typename T>
__device__ __forceinline__ void psi_gradient(const typename Pair<T>::type *__restrict__ psi, int n, const Nbr &o,
                                             T (&SA)[3], T (&SB)[3]) {
    T axA[3] = {T(0), T(0), T(0)}, dgA[3] = {T(0), T(0), T(0)};
    T axB[3] = {T(0), T(0), T(0)}, dgB[3] = {T(0), T(0), T(0)};
#pragma unroll
    for (int i = 1; i < L::Q; i++) {
        const typename Pair<T>::type p = __ldg(psi + (n + shift<L>(i, +1, o)));
        const bool axis = (L::ex(i) != 0) + (L::ey(i) != 0) + (L::ez(i) != 0) == 1;
        T(&a)[3] = axis ? axA : dgA;
        T(&b)[3] = axis ? axB : dgB;
        if (L::ex(i) == 1) { a[0] += p.x; b[0] += p.y; } else if (L::ex(i) == -1) { a[0] -= p.x; b[0] -= p.y; }
        if (L::ey(i) == 1) { a[1] += p.x; b[1] += p.y; } else if (L::ey(i) == -1) { a[1] -= p.x; b[1] -= p.y; }
        if (L::ez(i) == 1) { a[2] += p.x; b[2] += p.y; } else if (L::ez(i) == -1) { a[2] -= p.x; b[2] -= p.y; }
    }
    // axis weight / diagonal weight = 4 (D2Q9: 1/9 vs 1/36) or 2 (D3Q19: 1/18 vs 1/36)
    const T ratio = L::template w<T>(1) / L::template w<T>(L::Q - 1), wd = L::template w<T>(L::Q - 1);
#pragma unroll
    for (int c = 0; c < 3; c++) {
        SA[c] = wd * (ratio * axA[c] + dgA[c]);
        SB[c] = wd * (ratio * axB[c] + dgB[c]);
    }
}

template <class L, typename T, int PSI, int FS>
__device__ __forceinline__ void sc_collide_with_gradient(T (&hA)[L::Q], T (&hB)[L::Q], const T (&SA)[3], const T (&SB)[3],
                                                         const Relax<T> &rpA, const Relax<T> &rpB, T G);

// Collision of both components at one node (rows a10-a11): moments, common velocity u',
// coupling forces (eq. 10, sign A11) + body force, Guo (A13) or EDM (A22) per component; node types
// FULLWAY / VELOCITY replace the collision of both components.
template <class L, typename T, int PSI, int FS>
__device__ __forceinline__ void sc_collide_node(T (&hA)[L::Q], T (&hB)[L::Q], uint32_t t,
                                                const typename Pair<T>::type *__restrict__ psi, int n, const Nbr &o,
                                                const Relax<T> &rpA, const Relax<T> &rpB, T G) {
    if (t & (NODE_FULLWAY | NODE_VELOCITY)) {
        if (t & NODE_FULLWAY) { fullway_reverse<L, T>(hA); fullway_reverse<L, T>(hB); }
        else { velocity_node<L, T>(hA, rpA.ubc); velocity_node<L, T>(hB, rpB.ubc); }
        return;
    }
    T SA[3], SB[3];
    psi_gradient<L, T>(psi, n, o, SA, SB);
    sc_collide_with_gradient<L, T, PSI, FS>(hA, hB, SA, SB, rpA, rpB, G);
}

// ... with S_A, S_B already summed (the V-node kernel sums them row by row for the whole pack).
template <class L, typename T, int PSI, int FS>
__device__ __forceinline__ void sc_collide_with_gradient(T (&hA)[L::Q], T (&hB)[L::Q], const T (&SA)[3], const T (&SB)[3],
                                                         const Relax<T> &rpA, const Relax<T> &rpB, T G) {
    T dA, dB, jA[3], jB[3];
    moments<L, T>(hA, dA, jA);
    moments<L, T>(hB, dB, jB);
    const T rA = T(1) + dA, rB = T(1) + dB;
    const T pA = psi_dev<T, PSI>(dA) + psi_one<T, PSI>(), pB = psi_dev<T, PSI>(dB) + psi_one<T, PSI>();
    const T inv_den = T(1) / (rA * rpA.inv_tau + rB * rpB.inv_tau);
    const T irA = T(0.5) / rA, irB = T(0.5) / rB;
    T vA[3], vB[3], mA[3], mB[3], FA[3], FB[3];
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const T up = (jA[a] * rpA.inv_tau + jB[a] * rpB.inv_tau) * inv_den;
        FA[a] = -G * pA * SB[a] + rA * rpA.g[a];
        FB[a] = -G * pB * SA[a] + rB * rpB.g[a];
        // Guo: v_s = u' + F_s / (2 rho_s) (A13); EDM: the bare common velocity u' (A22)
        vA[a] = FS == FORCE_EDM ? up : up + FA[a] * irA;
        vB[a] = FS == FORCE_EDM ? up : up + FB[a] * irB;
        mA[a] = rA * vA[a];
        mB[a] = rB * vB[a];
    }
    collide<L, T, MODEL_BGK, FS>(hA, rA, dA, vA, mA, FA, rpA);
    collide<L, T, MODEL_BGK, FS>(hB, rB, dB, vB, mB, FB, rpB);
}

// S_A, S_B for the V nodes of a pack, summed row by row: for each of the (e_y, e_z) rows the D3Q19 / D2Q9
// neighbourhood touches, the interleaved field is read once for the whole pack (x0 - 1, the pack's own V
// columns as one aligned vector, x0 + V) instead of once per node and link: 19 loads per 2-node pack
// where the one-node kernel issues 36, all but the two edge columns 16 bytes wide.
template <typename T, int V> struct PairRow;
template <> struct PairRow<float, 2> {
    static __device__ __forceinline__ void ld(const float2 *p, float2 (&v)[2]) {
        const float4 q = __ldg(reinterpret_cast<const float4 *>(p));
        v[0] = make_float2(q.x, q.y); v[1] = make_float2(q.z, q.w);
    }
};
template <typename T> struct PairRow<T, 1> {
    static __device__ __forceinline__ void ld(const typename Pair<T>::type *p, typename Pair<T>::type (&v)[1]) { v[0] = __ldg(p); }
};
template <> struct PairRow<double, 2> {
    static __device__ __forceinline__ void ld(const double2 *p, double2 (&v)[2]) { v[0] = __ldg(p); v[1] = __ldg(p + 1); }
};

template <class L, typename T, int V>
__device__ __forceinline__ void psi_gradient_span(const typename Pair<T>::type *__restrict__ psi, const Span &s,
                                                  T (&SA)[V][3], T (&SB)[V][3]) {
    using P = typename Pair<T>::type;
    T axA[V][3], dgA[V][3], axB[V][3], dgB[V][3];
#pragma unroll
    for (int k = 0; k < V; k++)
#pragma unroll
        for (int c = 0; c < 3; c++) axA[k][c] = dgA[k][c] = axB[k][c] = dgB[k][c] = T(0);
#pragma unroll
    for (int dz = -1; dz <= 1; dz++) {
#pragma unroll
        for (int dy = -1; dy <= 1; dy++) {
            // which columns of row (dy, dz) the neighbourhood touches
            bool centre = false, sides = false;
#pragma unroll
            for (int i = 1; i < L::Q; i++)
                if (L::ey(i) == dy && L::ez(i) == dz) { if (L::ex(i) == 0) centre = true; else sides = true; }
            if (!centre && !sides) continue;
            const int r = s.row + (dy == 1 ? s.o.yp : dy == -1 ? s.o.ym : 0) + (dz == 1 ? s.o.zp : dz == -1 ? s.o.zm : 0);
            P v[V + 2];
            if (centre || V > 1) {  // the pack's own columns: neighbours at e_x = 0, and at e_x = +-1 of the other nodes
                P mid[V];
                PairRow<T, V>::ld(psi + (r + s.x0), mid);
#pragma unroll
                for (int k = 0; k < V; k++) v[k + 1] = mid[k];
            }
            if (sides) { v[0] = __ldg(psi + (r + s.xm)); v[V + 1] = __ldg(psi + (r + s.xp)); }
#pragma unroll
            for (int i = 1; i < L::Q; i++) {
                if (L::ey(i) != dy || L::ez(i) != dz) continue;
                const bool axis = (L::ex(i) != 0) + (dy != 0) + (dz != 0) == 1;
#pragma unroll
                for (int k = 0; k < V; k++) {
                    const P p = v[k + 1 + L::ex(i)];
                    T(&a)[3] = axis ? axA[k] : dgA[k];
                    T(&b)[3] = axis ? axB[k] : dgB[k];
                    if (L::ex(i) == 1) { a[0] += p.x; b[0] += p.y; } else if (L::ex(i) == -1) { a[0] -= p.x; b[0] -= p.y; }
                    if (dy == 1) { a[1] += p.x; b[1] += p.y; } else if (dy == -1) { a[1] -= p.x; b[1] -= p.y; }
                    if (dz == 1) { a[2] += p.x; b[2] += p.y; } else if (dz == -1) { a[2] -= p.x; b[2] -= p.y; }
                }
            }
        }
    }
    const T ratio = L::template w<T>(1) / L::template w<T>(L::Q - 1), wd = L::template w<T>(L::Q - 1);
#pragma unroll
    for (int k = 0; k < V; k++)
#pragma unroll
        for (int c = 0; c < 3; c++) {
            SA[k][c] = wd * (ratio * axA[k][c] + dgA[k][c]);
            SB[k][c] = wd * (ratio * axB[k][c] + dgB[k][c]);
        }
}

// Pass 2 (rows a10-a11): both components in one kernel: gather, moments, common velocity u'
// (P:188), forces (eq. 10, sign A11) + body force, v_s = u' + F_s / (2 rho_s), LBGK + Guo (A13).
template <class L, typename T, int V, typename I, int PSI, int FS>
__global__ void __launch_bounds__(256)
sc_step_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
               const T *__restrict__ srcA, const T *__restrict__ srcB, T *__restrict__ dstA,
               T *__restrict__ dstB, const typename Pair<T>::type *__restrict__ psi,
               Relax<T> rpA, Relax<T> rpB, T G) {
    Span s;
    if (!thread_span<V>(g, s)) return;
    const int n0 = s.row + s.x0;
    const uint32_t types = load_types<V>(type, n0);
    if (all_solid<V>(types)) return;
    T hA[V][L::Q], hB[V][L::Q];
    gather_span<L, T, V, I>(srcA, g.N, s, hA);
    gather_span<L, T, V, I>(srcB, g.N, s, hB);
    pull_reflected_span<L, T, V, I>(srcA, g.N, n0, types, link, hA);
    pull_reflected_span<L, T, V, I>(srcB, g.N, n0, types, link, hB);
    T SA[V][3], SB[V][3];
    psi_gradient_span<L, T, V>(psi, s, SA, SB);
#pragma unroll
    for (int k = 0; k < V; k++) {
        const uint32_t t = (types >> (8 * k)) & 0xffu;
        if (t & NODE_FULLWAY) { fullway_reverse<L, T>(hA[k]); fullway_reverse<L, T>(hB[k]); }
        else if (t & NODE_VELOCITY) { velocity_node<L, T>(hA[k], rpA.ubc); velocity_node<L, T>(hB[k], rpB.ubc); }
        else sc_collide_with_gradient<L, T, PSI, FS>(hA[k], hB[k], SA[k], SB[k], rpA, rpB, G);
    }
    store_span<L, T, V, I>(dstA, g.N, n0, hA);
    store_span<L, T, V, I>(dstB, g.N, n0, hB);
}


// ---- Shan-Chen, split variant ("split" kernels, one launch per component) -----------
// The paper found per-component collide kernels faster than one monolithic kernel by 5-53 % because of
// their smaller register footprint.  Same on B200: the monolithic kernel holds two components per node
// (80 registers at ONE node per thread, 70 % of the DRAM peak), a one-component kernel is the ordinary
// step kernel at V = 4 plus a force.  Price: the common velocity u' has to travel through memory.
//   pass 1  sc_fields_split_kernel: psi_A, psi_B (planar) and u' from the time-t state     152 B read, 20 B written (fp32)
//   pass 2  sc_collide_split_kernel, once per component s: pull f_s, S = sum_i w_i psi_other(x + e_i) e_i,
//           u', F_s, collide, store                                                         2 x (76 + 4 + 12 B read, 76 B written)
// 508 B per site instead of 472; which variant runs is chosen by measurement (lbm_b200.cu).
template <class L, typename T, int V, typename I, int PSI>
__global__ void __launch_bounds__(256)
sc_fields_split_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                       const T *__restrict__ srcA, const T *__restrict__ srcB, T *__restrict__ psiA,
                       T *__restrict__ psiB, T *__restrict__ up, T inv_tauA, T inv_tauB) {
    Span s;
    if (!thread_span<V>(g, s)) return;
    const int n0 = s.row + s.x0;
    const uint32_t types = load_types<V>(type, n0);
    T pa[V], pb[V], u[3][V];
#pragma unroll
    for (int k = 0; k < V; k++) { pa[k] = pb[k] = -psi_one<T, PSI>(); u[0][k] = u[1][k] = u[2][k] = T(0); }
    if (!all_solid<V>(types)) {
        T h[V][L::Q], rA[V], jA[V][3];
        gather_span<L, T, V, I>(srcA, g.N, s, h);
        pull_reflected_span<L, T, V, I>(srcA, g.N, n0, types, link, h);
#pragma unroll
        for (int k = 0; k < V; k++) {
            T d;
            moments<L, T>(h[k], d, jA[k]);
            rA[k] = T(1) + d;
            pa[k] = psi_dev<T, PSI>(d);
        }
        gather_span<L, T, V, I>(srcB, g.N, s, h);
        pull_reflected_span<L, T, V, I>(srcB, g.N, n0, types, link, h);
#pragma unroll
        for (int k = 0; k < V; k++) {
            T d, jB[3];
            moments<L, T>(h[k], d, jB);
            const T rB = T(1) + d;
            pb[k] = psi_dev<T, PSI>(d);
            const T inv_den = T(1) / (rA[k] * inv_tauA + rB * inv_tauB);
#pragma unroll
            for (int a = 0; a < 3; a++) u[a][k] = (jA[k][a] * inv_tauA + jB[a] * inv_tauB) * inv_den;  // u'
            if ((types >> (8 * k)) & (NODE_SOLID | NODE_FULLWAY)) {  // dry: psi = 0 (A14), no velocity
                pa[k] = pb[k] = -psi_one<T, PSI>();
                u[0][k] = u[1][k] = u[2][k] = T(0);
            }
        }
    }
    Pack<T, V>::stp(psiA + n0, pa);  // plain stores: pass 2 re-reads the fields right away (L2)
    Pack<T, V>::stp(psiB + n0, pb);
#pragma unroll
    for (int a = 0; a < L::D; a++) Pack<T, V>::stp(up + ((int64_t)a * g.N + n0), u[a]);
}

// S = sum_i w_i psi(x + e_i) e_i of ONE planar field for the V nodes of a pack, row by row (see psi_gradient_span).
template <class L, typename T, int V>
__device__ __forceinline__ void field_gradient_span(const T *__restrict__ psi, const Span &s, T (&S)[V][3]) {
    T ax[V][3], dg[V][3];
#pragma unroll
    for (int k = 0; k < V; k++)
#pragma unroll
        for (int c = 0; c < 3; c++) ax[k][c] = dg[k][c] = T(0);
#pragma unroll
    for (int dz = -1; dz <= 1; dz++) {
#pragma unroll
        for (int dy = -1; dy <= 1; dy++) {
            bool centre = false, sides = false;
#pragma unroll
            for (int i = 1; i < L::Q; i++)
                if (L::ey(i) == dy && L::ez(i) == dz) { if (L::ex(i) == 0) centre = true; else sides = true; }
            if (!centre && !sides) continue;
            const int r = s.row + (dy == 1 ? s.o.yp : dy == -1 ? s.o.ym : 0) + (dz == 1 ? s.o.zp : dz == -1 ? s.o.zm : 0);
            T v[V + 2];
            if (centre || V > 1) {
                T mid[V];
                Pack<T, V>::ld(psi + (r + s.x0), mid);
#pragma unroll
                for (int k = 0; k < V; k++) v[k + 1] = mid[k];
            }
            if (sides) { v[0] = __ldg(psi + (r + s.xm)); v[V + 1] = __ldg(psi + (r + s.xp)); }
#pragma unroll
            for (int i = 1; i < L::Q; i++) {
                if (L::ey(i) != dy || L::ez(i) != dz) continue;
                const bool axis = (L::ex(i) != 0) + (dy != 0) + (dz != 0) == 1;
#pragma unroll
                for (int k = 0; k < V; k++) {
                    const T p = v[k + 1 + L::ex(i)];
                    T(&a)[3] = axis ? ax[k] : dg[k];
                    if (L::ex(i) == 1) a[0] += p; else if (L::ex(i) == -1) a[0] -= p;
                    if (dy == 1) a[1] += p; else if (dy == -1) a[1] -= p;
                    if (dz == 1) a[2] += p; else if (dz == -1) a[2] -= p;
                }
            }
        }
    }
    const T ratio = L::template w<T>(1) / L::template w<T>(L::Q - 1), wd = L::template w<T>(L::Q - 1);
#pragma unroll
    for (int k = 0; k < V; k++)
#pragma unroll
        for (int c = 0; c < 3; c++) S[k][c] = wd * (ratio * ax[k][c] + dg[k][c]);
}

// One component's collision for the V nodes of a pack: S = gradient sum of the OTHER component's psi,
// u = common velocity u' (component planes).  Node types FULLWAY / VELOCITY replace the collision.
template <class L, typename T, int V, int PSI, int FS>
__device__ __forceinline__ void sc_component_update_span(T (&h)[V][L::Q], uint32_t types, const T (&S)[V][3],
                                                         const T (&u)[3][V], const Relax<T> &rp, T G) {
#pragma unroll
    for (int k = 0; k < V; k++) {
        const uint32_t t = (types >> (8 * k)) & 0xffu;
        if (t & NODE_FULLWAY) fullway_reverse<L, T>(h[k]);
        else if (t & NODE_VELOCITY) velocity_node<L, T>(h[k], rp.ubc);
        else {
            T d, j[3];
            moments<L, T>(h[k], d, j);
            const T r = T(1) + d, p = psi_dev<T, PSI>(d) + psi_one<T, PSI>(), ir = T(0.5) / r;
            T v[3], m[3], F[3];
#pragma unroll
            for (int a = 0; a < 3; a++) {
                F[a] = -G * p * S[k][a] + r * rp.g[a];               // eq. (10), sign A11, + body force
                v[a] = FS == FORCE_EDM ? u[a][k] : u[a][k] + F[a] * ir;  // Guo: v_s = u' + F_s / (2 rho_s) (A13); EDM: u' (A22)
                m[a] = r * v[a];
            }
            collide<L, T, MODEL_BGK, FS>(h[k], r, d, v, m, F, rp);
        }
    }
}

template <class L, typename T, int V>
__device__ __forceinline__ void load_common_velocity(const T *__restrict__ up, int64_t N, int n0, T (&u)[3][V]) {
#pragma unroll
    for (int a = 0; a < 3; a++) {
        if (a < L::D) Pack<T, V>::ldp(up + ((int64_t)a * N + n0), u[a]);
        else {
#pragma unroll
            for (int k = 0; k < V; k++) u[a][k] = T(0);
        }
    }
}

template <class L, typename T, int V, typename I, int PSI, int FS>
__global__ void __launch_bounds__(256)
sc_collide_split_kernel(Geom g, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                        const T *__restrict__ src, T *__restrict__ dst, const T *__restrict__ psi_other,
                        const T *__restrict__ up, Relax<T> rp, T G) {
    Span s;
    if (!thread_span<V>(g, s)) return;
    const int n0 = s.row + s.x0;
    const uint32_t types = load_types<V>(type, n0);
    if (all_solid<V>(types)) return;
    T h[V][L::Q];
    gather_span<L, T, V, I>(src, g.N, s, h);
    T u[3][V];
    load_common_velocity<L, T, V>(up, g.N, n0, u);
    T S[V][3];
    field_gradient_span<L, T, V>(psi_other, s, S);
    pull_reflected_span<L, T, V, I>(src, g.N, n0, types, link, h);
    sc_component_update_span<L, T, V, PSI, FS>(h, types, S, u, rp, G);
    store_span<L, T, V, I>(dst, g.N, n0, h);
}

// ---- Shan-Chen on the in-place AA store: the split variant on both parities ---------------------
// Pass 1 reads f_A, f_B where the current parity keeps them (even: (i, x); odd: see aa_gather_odd_span)
// and writes psi_A, psi_B, u'; pass 2 is the AA even / odd step of ONE component with the coupling force.
template <class L, typename T, int V, typename I>
__device__ __forceinline__ void aa_gather_span(int parity, const T *f, const Geom &g, const Span &s, uint32_t types,
                                               const uint32_t *__restrict__ link, T (&h)[V][L::Q]) {
    if (parity == 0) {
#pragma unroll
        for (int i = 0; i < L::Q; i++) {
            T a[V];
            Pack<T, V>::ldp(f + (I(i) * I(g.N) + I(s.row + s.x0)), a);
#pragma unroll
            for (int k = 0; k < V; k++) h[k][i] = a[k];
        }
    } else {
        aa_gather_odd_span<L, T, V, I>(f, g, s, types, link, h);
    }
}

template <class L, typename T, int V, typename I, int PSI>
__global__ void __launch_bounds__(256)
aa_sc_fields_split_kernel(Geom g, int parity, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link,
                          const T *fA, const T *fB, T *__restrict__ psiA, T *__restrict__ psiB, T *__restrict__ up,
                          T inv_tauA, T inv_tauB) {
    Span s;
    if (!thread_span<V>(g, s)) return;
    const int n0 = s.row + s.x0;
    const uint32_t types = load_types<V>(type, n0);
    T pa[V], pb[V], u[3][V];
#pragma unroll
    for (int k = 0; k < V; k++) { pa[k] = pb[k] = -psi_one<T, PSI>(); u[0][k] = u[1][k] = u[2][k] = T(0); }
    if (!all_solid<V>(types)) {
        T h[V][L::Q], rA[V], jA[V][3];
        aa_gather_span<L, T, V, I>(parity, fA, g, s, types, link, h);
#pragma unroll
        for (int k = 0; k < V; k++) {
            T d;
            moments<L, T>(h[k], d, jA[k]);
            rA[k] = T(1) + d;
            pa[k] = psi_dev<T, PSI>(d);
        }
        aa_gather_span<L, T, V, I>(parity, fB, g, s, types, link, h);
#pragma unroll
        for (int k = 0; k < V; k++) {
            T d, jB[3];
            moments<L, T>(h[k], d, jB);
            const T rB = T(1) + d;
            pb[k] = psi_dev<T, PSI>(d);
            const T inv_den = T(1) / (rA[k] * inv_tauA + rB * inv_tauB);
#pragma unroll
            for (int a = 0; a < 3; a++) u[a][k] = (jA[k][a] * inv_tauA + jB[a] * inv_tauB) * inv_den;
            if ((types >> (8 * k)) & (NODE_SOLID | NODE_FULLWAY)) {
                pa[k] = pb[k] = -psi_one<T, PSI>();
                u[0][k] = u[1][k] = u[2][k] = T(0);
            }
        }
    }
    Pack<T, V>::stp(psiA + n0, pa);
    Pack<T, V>::stp(psiB + n0, pb);
#pragma unroll
    for (int a = 0; a < L::D; a++) Pack<T, V>::stp(up + ((int64_t)a * g.N + n0), u[a]);
}

template <class L, typename T, int V, typename I, int PSI, int FS>
__global__ void __launch_bounds__(AA_MAX_BLOCK)
aa_sc_collide_split_kernel(Geom g, int parity, const uint8_t *__restrict__ type, const uint32_t *__restrict__ link, T *f,
                           const T *__restrict__ psi_other, const T *__restrict__ up, Relax<T> rp, T G) {
    Span s;
    const bool valid = thread_span_all<V>(g, s);
    const int n0 = s.row + s.x0;
    const uint32_t types = valid ? load_types<V>(type, n0) : PACK_SOLID;
    const bool live = valid && !all_solid<V>(types);
    T h[V][L::Q];
    if (live) {
        aa_gather_span<L, T, V, I>(parity, f, g, s, types, link, h);
        T u[3][V], S[V][3];
        load_common_velocity<L, T, V>(up, g.N, n0, u);
        field_gradient_span<L, T, V>(psi_other, s, S);
        sc_component_update_span<L, T, V, PSI, FS>(h, types, S, u, rp, G);
    }
    if (parity == 0) {  // even: local, h*_i to (ibar, x)
        if (live) {
#pragma unroll
            for (int i = 0; i < L::Q; i++) {
                T a[V];
#pragma unroll
                for (int k = 0; k < V; k++) a[k] = h[k][i];
                Pack<T, V>::stp(f + (I(L::opp(i)) * I(g.N) + I(n0)), a);
            }
        }
    } else {
        aa_scatter_odd_span<L, T, V, I>(f, g, s, types, live, link, h);
    }
}

}  // namespace lbm
