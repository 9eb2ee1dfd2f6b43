// m2p_inst.cu -- one translation unit per expansion order: nvcc -DM2P_P=<P>.
#include "m2p.cuh"
#ifndef M2P_P
#error "compile with -DM2P_P=<order>"
#endif
#define CAT_(a, b) a##b
#define CAT(a, b) CAT_(a, b)

#ifdef M2P_STUB
int CAT(pygbe_m2p_launch_, M2P_P)(const M2PArgs &) { return -1; }
#else
template <bool TWIN, typename T> static void launch(const M2PArgs &a)
{
    k_m2p<M2P_P, TWIN, T><<<a.n_items, PYGBE_TG_M2P, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.cgeo,
                                                                    (const T *)a.wc, a.kappaA, Real<T>::kscale(a.kappaA),
                                                                    a.kappaB, Real<T>::kscale(a.kappaB), a.outA, a.outB);
}

int CAT(pygbe_m2p_launch_, M2P_P)(const M2PArgs &a)
{
    if (a.lap && a.fp32) {                // kappa = 0, no twin: one polynomial in d / r^2 by Horner steps, four targets per thread
        k_m2p_lap<M2P_P, float><<<a.n_items, M2PL_THREADS, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.ggeo, a.cgeo,
                                                                          (const float *)a.wc, a.outA);
    } else if (a.lap) {
        k_m2p_lap<M2P_P, double><<<a.n_items, M2PL_THREADS, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.ggeo, a.cgeo,
                                                                           (const double *)a.wc, a.outA);
    } else if (a.fp32 && a.twin) {        // two targets per thread, packed fp32
        k_m2p_twin2<M2P_P><<<a.n_items, M2P2_THREADS, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.cgeo, (const float *)a.wc,
                                                                  a.kappaA, Real<float>::kscale(a.kappaA), a.kappaB,
                                                                  Real<float>::kscale(a.kappaB), a.outA, a.outB);
    } else if (a.fp32) {
        k_m2p_single2<M2P_P><<<a.n_items, M2P2_THREADS, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.cgeo, (const float *)a.wc,
                                                                    a.kappaA, Real<float>::kscale(a.kappaA), a.outA);
    }
#if M2P_P <= 7
    else if (a.twin) {                    // fp64, two targets per thread: 0.156 -> 0.145 ms at P = 6 (config 1)
        k_m2p_dbl2<M2P_P, true><<<a.n_items, M2P2_THREADS, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.cgeo,
                                                                       (const double *)a.wc, a.kappaA, a.kappaB, a.outA, a.outB);
    } else {
        k_m2p_dbl2<M2P_P, false><<<a.n_items, M2P2_THREADS, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.cgeo,
                                                                        (const double *)a.wc, a.kappaA, a.kappaB, a.outA, a.outB);
    }
#else                                     // P >= 8: 158+ registers with two targets, no gain (1.344 against 1.331 ms at P = 8)
    else { if (a.twin) launch<true, double>(a); else launch<false, double>(a); }
#endif
    return 0;
}
#endif
