// Host-compiled unit check of the product's per-node arithmetic (csrc/lbm_node.cuh), built by
// tests/test_node_math_host.py with g++.  TEST ONLY: lets the CPU suite compare the collision
// templates with the oracle on a 1x1x1 torus (where streaming is the identity) without a GPU.
// It is not a CPU fallback: nothing in the package builds, loads or calls it.
#include "../paper_1311_2404_b200/csrc/lbm_node.cuh"

using namespace lbm;

template <class L, typename T, int MODEL, int FORCE>
static void run(const double *f, double tau, const double *rates, const double *g, double *out, double cs = 0.0) {
    Relax<T> rp{};
    set_bgk(rp, tau);
    for (int a = 0; a < 3; a++) rp.g[a] = T(g[a]);
    for (int k = 0; k < L::Q; k++) {
        rp.cr[k] = T(rates[k] / Mrt<L, double>::norm(k));
        rp.cs[k] = T((1.0 - 0.5 * rates[k]) / Mrt<L, double>::norm(k));
        rp.in[k] = T(1.0 / Mrt<L, double>::norm(k));
    }
    T h[L::Q];
    for (int i = 0; i < L::Q; i++) h[i] = T(f[i] - L::template w<double>(i));
    rp.cs2x36 = T(36.0 * cs * cs);
    update_node<L, T, MODEL, FORCE>(h, rp);
    for (int i = 0; i < L::Q; i++) out[i] = double(h[i]) + L::template w<double>(i);
}

template <class L, typename T>
static void dispatch(int mrt, int force, const double *f, double tau, const double *rates, const double *g, double *out) {
    // force: 0 none, 1 Guo (eq. 17), 2 Exact Difference Method (eq. 18)
    // mrt = model: 0 LBGK, 1 MRT, 2 regularized LBGK, 3 LBGK + Smagorinsky (C_S = 0.17 here)
    if (mrt == 1) {
        if (force == 2) run<L, T, 1, 2>(f, tau, rates, g, out);
        else if (force) run<L, T, 1, 1>(f, tau, rates, g, out);
        else run<L, T, 1, 0>(f, tau, rates, g, out);
    } else if (mrt == 2) {
        if (force == 2) run<L, T, 2, 2>(f, tau, rates, g, out);
        else run<L, T, 2, 0>(f, tau, rates, g, out);
    } else if (mrt == 3) {
        if (force == 2) run<L, T, 3, 2>(f, tau, rates, g, out, 0.17);
        else if (force) run<L, T, 3, 1>(f, tau, rates, g, out, 0.17);
        else run<L, T, 3, 0>(f, tau, rates, g, out, 0.17);
    } else {
        if (force == 2) run<L, T, 0, 2>(f, tau, rates, g, out);
        else if (force) run<L, T, 0, 1>(f, tau, rates, g, out);
        else run<L, T, 0, 0>(f, tau, rates, g, out);
    }
}

extern "C" int host_update_node(int lattice, int f32, int mrt, int force, const double *f, double tau,
                                const double *rates, const double *g, double *out) {
    if (lattice == 0) { if (f32) dispatch<D2Q9, float>(mrt, force, f, tau, rates, g, out); else dispatch<D2Q9, double>(mrt, force, f, tau, rates, g, out); }
    else              { if (f32) dispatch<D3Q19, float>(mrt, force, f, tau, rates, g, out); else dispatch<D3Q19, double>(mrt, force, f, tau, rates, g, out); }
    return 0;
}

// M d and M^T r for the MRT pin (row-by-row comparison with the oracle's matrix)
extern "C" int host_mrt_transform(int lattice, int backward, const double *in, double *out) {
    if (lattice == 0) {
        double a[9], b[9];
        for (int i = 0; i < 9; i++) a[i] = in[i];
        if (backward) Mrt<D2Q9, double>::backward(a, b); else Mrt<D2Q9, double>::forward(a, b);
        for (int i = 0; i < 9; i++) out[i] = b[i];
    } else {
        double a[19], b[19];
        for (int i = 0; i < 19; i++) a[i] = in[i];
        if (backward) Mrt<D3Q19, double>::backward(a, b); else Mrt<D3Q19, double>::forward(a, b);
        for (int i = 0; i < 19; i++) out[i] = b[i];
    }
    return 0;
}
