// m2p_inst.cu -- one translation unit per expansion order: nvcc -DM2P_P=<P>.
#include "m2p.cuh"
#ifndef M2P_P
#error "compile with -DM2P_P=<order>"
#endif
#define CAT_(a, b) a##b
#define CAT(a, b) CAT_(a, b)

int CAT(pygbe_m2p_f64_launch_, M2P_P)(const M2PArgs &a)
{
    if (a.yukawa)
        k_m2p_f64<M2P_P, true><<<a.n_items, PYGBE_TG_M2P, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.cgeo,
                                                                        a.mom, a.kappa, a.out);
    else
        k_m2p_f64<M2P_P, false><<<a.n_items, PYGBE_TG_M2P, 0, a.stream>>>(a.skip, a.items, a.m2p_cell, a.np, a.tpos, a.cgeo,
                                                                         a.mom, a.kappa, a.out);
    return 0;
}
