// mma_probe.cuh -- the tensor-core question of the north star, answered with numbers (SURVEY 8(d) "Tensor cores",
// 8(f) item 3): "tensor cores are used only if a batched M2P stage is shown to be a dense contraction".
//
// In the regrouped form of the series (m2p.cuh; harmonically reduced moments, Ne = (P+1)^2 monomials with ez <= 1) the
// 64 targets of a group multiply their monomial rows d^e by the SAME per-cell coefficients: per (group, cell) that is
// the product  Q[64 x (P+1)] = A[64 x Ne] * B[Ne x (P+1)],
// A[t][e] = d_t^e (target-specific, recomputed for every cell), B[e][m] = W_{m,e} (23 % dense), followed by
// sum_m F^(m)(r_t) Q[t][m].  This file measures, on synthetic far-field data shaped like the M2P lists of the Yukawa
// region of config 4 (P = 8, single moment set, 64-target groups, cells of 2-8 A at 1.1-3 times the MAC distance),
//   cuda   the production kernel k_m2p_single2<P> (packed fp32 FMAs, coefficients broadcast from shared memory),
//   tile   only what ANY tensor-core formulation has to do first: put the 64 x Ne monomial tile of every (group,
//          cell) into shared memory (tcgen05.mma and mma.sync both read A from shared memory / TMEM, and the
//          monomials are per target and per cell, so the tile cannot be reused or loaded by TMA),
//   mma1   tile + the contraction on the tensor cores in one TF32 pass + the radial combination,
//   mma3   the same with the 3 x TF32 split (A = A_hi + A_lo, B = B_hi + B_lo; hi*hi + hi*lo + lo*hi),
// each with its relative L2 error against fp64 direct sums.  The contraction is issued as mma.sync.m16n8k8.tf32
// (it runs on the same tensor cores; tcgen05.mma would shorten only the MMA part -- the table shows that the
// tile alone already costs more than the whole CUDA-core evaluation, so the issue path does not decide).
// Nothing here is on the product path; bench.py --probe-mma prints the table (profiles/r4_m2p_mma.md).
#pragma once
#include <random>
#include "common.cuh"
#include "tables.cuh"
#include "m2p.cuh"

#define MP_TG 64
__device__ __forceinline__ float to_tf32(float x)
{
    unsigned u;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(u) : "f"(x));
    return __uint_as_float(u);
}
__device__ __forceinline__ void mma_tf32(float (&d)[4], const float (&a)[4], const float (&b)[2])
{
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(__float_as_uint(a[0])), "r"(__float_as_uint(a[1])), "r"(__float_as_uint(a[2])), "r"(__float_as_uint(a[3])),
                   "r"(__float_as_uint(b[0])), "r"(__float_as_uint(b[1])));
}

template <int P> struct MmaShape {
    static constexpr int NC = (P + 1) * (P + 1);           // monomials d^e of the reduced index set (ez <= 1)
    static constexpr int KP = (NC + 7) / 8 * 8;            // K padded to the MMA's k = 8
    static constexpr int NP = (P + 1 + 7) / 8 * 8;         // N padded to n = 8 tiles
    static constexpr int AS = KP + 1;                      // row stride of the A tile (odd: conflict-free row writes)
    static constexpr int BS = KP + 4;                      // row stride of the B tile [n][k]
};

// one warp per group: lanes own targets lane and lane + 32; the monomials of both go to rows lane, lane + 32 of the
// tile in the order of m2p_q (ex, ey, ez ascending); SPLIT also writes the tf32 remainder tile
template <int P, bool SPLIT>
__device__ __forceinline__ void mp_build_tile(float dx0, float dy0, float dz0, float dx1, float dy1, float dz1, int lane,
                                              float *__restrict__ sA, float *__restrict__ sAlo)
{
    typedef MmaShape<P> S;
    float *r0 = sA + lane * S::AS, *r1 = sA + (lane + 32) * S::AS;
    float *l0 = sAlo + lane * S::AS, *l1 = sAlo + (lane + 32) * S::AS;
    int idx = 0;
    float px0 = 1.f, px1 = 1.f;
#pragma unroll
    for (int ex = 0; ex <= P; ex++) {
        float pxy0 = px0, pxy1 = px1;
#pragma unroll
        for (int ey = 0; ey <= P - ex; ey++) {
            float m0 = pxy0, m1 = pxy1;
#pragma unroll
            for (int ez = 0; ez <= M2P_EZ(P, ex, ey); ez++) {
                const float h0 = to_tf32(m0), h1 = to_tf32(m1);
                r0[idx] = h0; r1[idx] = h1;
                if (SPLIT) { l0[idx] = to_tf32(m0 - h0); l1[idx] = to_tf32(m1 - h1); }
                idx++;
                m0 *= dz0; m1 *= dz1;
            }
            pxy0 *= dy0; pxy1 *= dy1;
        }
        px0 *= dx0; px1 *= dx1;
    }
#pragma unroll
    for (int k = S::NC; k < S::KP; k++) { r0[k] = 0.f; r1[k] = 0.f; if (SPLIT) { l0[k] = 0.f; l1[k] = 0.f; } }
}

// MODE 0: tile only (a checksum of the tile keeps the stores alive); 1: one TF32 pass; 3: 3 x TF32
template <int P, int MODE>
__global__ void __launch_bounds__(32)
k_mp_mma(int n_groups, int cells_per_group, const int *__restrict__ cell_of, const double4 *__restrict__ tpos,
         const double4 *__restrict__ cgeo, const float *__restrict__ Bhi, const float *__restrict__ Blo, double kappa,
         double *__restrict__ out)
{
    typedef MmaShape<P> S;
    constexpr bool SPLIT = MODE == 3;
    extern __shared__ float s_mp[];
    float *sA = s_mp, *sAlo = sA + (SPLIT ? MP_TG * S::AS : 0);
    float *sB = sAlo + MP_TG * S::AS, *sBlo = sB + (SPLIT ? S::NP * S::BS : 0);
    const int g = blockIdx.x, lane = threadIdx.x, gid = lane >> 2, tig = lane & 3;
    if (g >= n_groups) return;
    const double4 X0 = tpos[g * MP_TG + lane], X1 = tpos[g * MP_TG + lane + 32];
    const float kap = (float)kappa, ks = (float)(kappa * 1.4426950408889634);
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};                          // rows gid + 8 j, j = 0..7 (partial over this lane's columns)
    double chk = 0.0;
    for (int c_ = 0; c_ < cells_per_group; c_++) {
        const int cell = cell_of[g * cells_per_group + c_];
        const double4 c = cgeo[cell];
        __syncwarp();
        mp_build_tile<P, SPLIT>((float)(X0.x - c.x), (float)(X0.y - c.y), (float)(X0.z - c.z), (float)(X1.x - c.x), (float)(X1.y - c.y),
                                (float)(X1.z - c.z), lane, sA, sAlo);
        if (MODE == 0) {
            __syncwarp();
            chk += sA[((lane * 7 + c_) % MP_TG) * S::AS + (lane + c_) % S::NC];
            continue;
        }
        for (int i = lane; i < S::NP * S::KP / 4; i += 32) {           // the cell's dense coefficient tile, [n][k]
            const int n = i / (S::KP / 4), k4 = i - n * (S::KP / 4);
            *(float4 *)(sB + n * S::BS + 4 * k4) = *(const float4 *)(Bhi + ((long)cell * S::NP + n) * S::KP + 4 * k4);
            if (SPLIT) *(float4 *)(sBlo + n * S::BS + 4 * k4) = *(const float4 *)(Blo + ((long)cell * S::NP + n) * S::KP + 4 * k4);
        }
        __syncwarp();
        float d[4][S::NP / 8][4];
#pragma unroll
        for (int mt = 0; mt < 4; mt++)
#pragma unroll
            for (int nt = 0; nt < S::NP / 8; nt++)
#pragma unroll
                for (int q = 0; q < 4; q++) d[mt][nt][q] = 0.f;
#pragma unroll 1
        for (int k0 = 0; k0 < S::KP; k0 += 8) {
            float b[S::NP / 8][2], bl[S::NP / 8][2];
#pragma unroll
            for (int nt = 0; nt < S::NP / 8; nt++) {
                b[nt][0] = sB[(nt * 8 + gid) * S::BS + k0 + tig]; b[nt][1] = sB[(nt * 8 + gid) * S::BS + k0 + tig + 4];
                if (SPLIT) { bl[nt][0] = sBlo[(nt * 8 + gid) * S::BS + k0 + tig]; bl[nt][1] = sBlo[(nt * 8 + gid) * S::BS + k0 + tig + 4]; }
            }
#pragma unroll
            for (int mt = 0; mt < 4; mt++) {
                float a[4], al[4];
                const float *ar = sA + (mt * 16 + gid) * S::AS + k0 + tig;
                a[0] = ar[0]; a[1] = ar[8 * S::AS]; a[2] = ar[4]; a[3] = ar[8 * S::AS + 4];
                if (SPLIT) { const float *lr = sAlo + (mt * 16 + gid) * S::AS + k0 + tig; al[0] = lr[0]; al[1] = lr[8 * S::AS]; al[2] = lr[4]; al[3] = lr[8 * S::AS + 4]; }
#pragma unroll
                for (int nt = 0; nt < S::NP / 8; nt++) {
                    mma_tf32(d[mt][nt], a, b[nt]);
                    if (SPLIT) { mma_tf32(d[mt][nt], a, bl[nt]); mma_tf32(d[mt][nt], al, b[nt]); }
                }
            }
        }
        // radial combination for the rows this lane holds: rows mt * 16 + gid (+ 8), columns m = nt * 8 + 2 tig (+ 1)
#pragma unroll
        for (int mt = 0; mt < 4; mt++)
#pragma unroll
            for (int hh = 0; hh < 2; hh++) {
                const int row = mt * 16 + gid + 8 * hh;
                const double4 X = tpos[g * MP_TG + row];
                const float dx = (float)(X.x - c.x), dy = (float)(X.y - c.y), dz = (float)(X.z - c.z);
                const float r2 = dx * dx + dy * dy + dz * dz;
                const float rinv = Real<float>::rsqrt_(r2), rinv2 = rinv * rinv, r = r2 * rinv;
                const float E = Real<float>::exp_neg(ks, r);
                float F[P + 1];
                F[0] = E * rinv;
                if (P >= 1) F[1] = -E * (kap * r + 1.f) * rinv * rinv2;
#pragma unroll
                for (int m = 1; m < P; m++) F[m + 1] = -((float)(2 * m + 1) * F[m] - kap * kap * F[m - 1]) * rinv2;
                float s = 0.f;
#pragma unroll
                for (int nt = 0; nt < S::NP / 8; nt++)
#pragma unroll
                    for (int q = 0; q < 2; q++) {
                        const int m = nt * 8 + 2 * tig + q;
                        if (m <= P) s = fmaf(F[m < P + 1 ? m : 0], d[mt][nt][2 * hh + q], s);
                    }
                acc[2 * mt + hh] += (double)s;
            }
    }
    if (MODE == 0) { if (chk == -1.2345) out[0] = chk; return; }
#pragma unroll
    for (int j = 0; j < 8; j++) {                                      // the four lanes of a quad hold the columns of a row
        double v = acc[j];
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        if (tig == 0) out[g * MP_TG + (j >> 1) * 16 + gid + 8 * (j & 1)] = v;
    }
}

// fp64 direct sums over the charges of the group's cells: the reference of the probe
__global__ void k_mp_direct(int n_groups, int cells_per_group, int nq, const int *__restrict__ cell_of, const double4 *__restrict__ tpos,
                            const double4 *__restrict__ qpos, double kappa, double *__restrict__ out)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_groups * MP_TG) return;
    const int g = t / MP_TG;
    const double4 X = tpos[t];
    double acc = 0.0;
    for (int c_ = 0; c_ < cells_per_group; c_++) {
        const int cell = cell_of[g * cells_per_group + c_];
        for (int k = 0; k < nq; k++) {
            const double4 q = qpos[(long)cell * nq + k];
            const double dx = X.x - q.x, dy = X.y - q.y, dz = X.z - q.z;
            const double r = sqrt(dx * dx + dy * dy + dz * dz);
            acc += q.w * exp(-kappa * r) / r;
        }
    }
    out[t] = acc;
}

int pygbe_m2p_launch_6(const M2PArgs &);
int pygbe_m2p_launch_8(const M2PArgs &);

// out[0..11]: ms and rel-L2 error vs fp64 direct sums of {cuda, tile, mma1, mma3}: out[3 v] = ms per launch,
// out[3 v + 1] = rel-L2 (NaN for the tile-only variant), out[3 v + 2] = (group, cell) pairs per launch
template <int P> static int run_mma_probe_p(int device, double *out)
{
    typedef MmaShape<P> S;
    CUDA_TRY(cudaSetDevice(device));
    const int G = 8192, C = 32, NCELL = 4096, NQ = 8;
    const double kappa = 0.125;
    std::mt19937_64 rng(13094018);
    std::uniform_real_distribution<double> U(0.0, 1.0);
    std::normal_distribution<double> N01(0.0, 1.0);
    auto unit = [&](double *v) { double n; do { v[0] = N01(rng); v[1] = N01(rng); v[2] = N01(rng); n = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]); } while (n < 1e-3); v[0] /= n; v[1] /= n; v[2] /= n; };
    // targets: groups of 64 points in 3 A cubes inside a ball of radius 10 A; cells: edge 2, 4 or 8 A, far enough from
    // that ball for the MAC theta = 0.5 (distance to the nearest possible target between 1.1 and 3 times edge / theta)
    std::vector<double4> tpos((size_t)G * MP_TG), cgeo(NCELL), qpos((size_t)NCELL * NQ);
    for (int g = 0; g < G; g++) {
        double d[3]; unit(d); const double rr = 8.0 * std::cbrt(U(rng));
        for (int t = 0; t < MP_TG; t++)
            tpos[(size_t)g * MP_TG + t] = make_double4(d[0] * rr + 3.0 * (U(rng) - 0.5), d[1] * rr + 3.0 * (U(rng) - 0.5), d[2] * rr + 3.0 * (U(rng) - 0.5), 0.0);
    }
    IndexTables *it = new IndexTables;
    fill_index_tables(it);
    WTable wt;
    build_w_table(P, kappa, *it, &wt);
    const int NW = (int)wt.off.size() - 1, stride = m2p_stride(P, false);
    std::vector<float> wc((size_t)NCELL * stride, 0.f), Bhi((size_t)NCELL * S::NP * S::KP, 0.f), Blo(Bhi.size(), 0.f);
    auto tf32 = [](float x) { unsigned u; memcpy(&u, &x, 4); u += 0x1000u; u &= 0xffffe000u; float y; memcpy(&y, &u, 4); return y; };   // round to nearest (ties away), 10-bit mantissa
    const int NCF = nc_of(P);                              // full set of Cartesian moments, the input of the table
    std::vector<double> M(NCF);
    for (int c = 0; c < NCELL; c++) {
        const double edge = 2.0 * (1 << (c % 3));
        double d[3]; unit(d);
        const double dist = 10.6 + edge / 0.5 * (1.1 + 1.9 * U(rng));
        cgeo[c] = make_double4(d[0] * dist, d[1] * dist, d[2] * dist, edge);
        std::fill(M.begin(), M.end(), 0.0);
        for (int k = 0; k < NQ; k++) {
            const double x = edge * (U(rng) - 0.5), y = edge * (U(rng) - 0.5), z = edge * (U(rng) - 0.5), q = N01(rng);
            qpos[(size_t)c * NQ + k] = make_double4(cgeo[c].x + x, cgeo[c].y + y, cgeo[c].z + z, q);
            for (int i = 0; i < NCF; i++)
                M[i] += q * std::pow(x, it->kxyz[i][0]) * std::pow(y, it->kxyz[i][1]) * std::pow(z, it->kxyz[i][2]);
        }
        // W stream (m2p.cuh order) and the same numbers as the dense tile B[m][e]
        int p = 0, e = 0;
        for (int ex = 0; ex <= P; ex++)
            for (int ey = 0; ey <= P - ex; ey++)
                for (int ez = 0; ez <= M2P_EZ(P, ex, ey); ez++, e++)
                    for (int J = 0; J <= (P - ex - ey - ez) / 2; J++, p++) {
                        double w = 0.0;
                        for (int i = wt.off[p]; i < wt.off[p + 1]; i++) w += wt.c[i] * M[wt.k[i]];
                        const float wf = (float)w;
                        wc[(size_t)c * stride + p] = wf;
                        const int m = ex + ey + ez + J;
                        const float hi = tf32(wf);
                        Bhi[((size_t)c * S::NP + m) * S::KP + e] = hi;
                        Blo[((size_t)c * S::NP + m) * S::KP + e] = tf32(wf - hi);
                    }
        if (p != NW) { delete it; pygbe_set_error("mma probe: table size mismatch"); return PYGBE_EINVAL; }
    }
    delete it;
    std::vector<int> cell_of((size_t)G * C);
    for (size_t i = 0; i < cell_of.size(); i++) cell_of[i] = (int)(rng() % NCELL);
    std::vector<int4> items(G);
    for (int g = 0; g < G; g++) items[g] = make_int4(g, g * C, (g + 1) * C, 0);

    double4 *d_tpos = nullptr, *d_cgeo = nullptr, *d_qpos = nullptr; float *d_wc = nullptr, *d_Bhi = nullptr, *d_Blo = nullptr;
    int *d_cell = nullptr; int4 *d_items = nullptr; double *d_out = nullptr, *d_ref = nullptr;
    auto up = [&](auto **dst, const auto &src) { cudaMalloc((void **)dst, src.size() * sizeof(src[0])); return cudaMemcpy(*dst, src.data(), src.size() * sizeof(src[0]), cudaMemcpyHostToDevice); };
    CUDA_TRY(up(&d_tpos, tpos)); CUDA_TRY(up(&d_cgeo, cgeo)); CUDA_TRY(up(&d_qpos, qpos)); CUDA_TRY(up(&d_wc, wc));
    CUDA_TRY(up(&d_Bhi, Bhi)); CUDA_TRY(up(&d_Blo, Blo)); CUDA_TRY(up(&d_cell, cell_of)); CUDA_TRY(up(&d_items, items));
    const size_t nt = (size_t)G * MP_TG;
    CUDA_TRY(cudaMalloc((void **)&d_out, nt * sizeof(double))); CUDA_TRY(cudaMalloc((void **)&d_ref, nt * sizeof(double)));
    k_mp_direct<<<cdiv((long)nt, 128), 128>>>(G, C, NQ, d_cell, d_tpos, d_qpos, kappa, d_ref);
    std::vector<double> ref(nt), got(nt);
    CUDA_TRY(cudaMemcpy(ref.data(), d_ref, nt * sizeof(double), cudaMemcpyDeviceToHost));
    double refn = 0.0;
    for (double v : ref) refn += v * v;
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0)); CUDA_TRY(cudaEventCreate(&e1));
    const size_t sm1 = ((size_t)MP_TG * S::AS + (size_t)S::NP * S::BS) * sizeof(float), sm3 = 2 * sm1, sm0 = (size_t)MP_TG * S::AS * sizeof(float);
    CUDA_TRY(cudaFuncSetAttribute(k_mp_mma<P, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm0));
    CUDA_TRY(cudaFuncSetAttribute(k_mp_mma<P, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm1));
    CUDA_TRY(cudaFuncSetAttribute(k_mp_mma<P, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm3));
    M2PArgs a;
    memset(&a, 0, sizeof(a));
    a.items = d_items; a.m2p_cell = d_cell; a.n_items = G; a.np = (int)nt; a.tpos = d_tpos; a.cgeo = d_cgeo; a.wc = d_wc;
    a.kappaA = kappa; a.outA = d_out; a.fp32 = 1;
    for (int v = 0; v < 4; v++) {
        float best = 1e30f;
        for (int rep = 0; rep < 6; rep++) {
            CUDA_TRY(cudaMemset(d_out, 0, nt * sizeof(double)));
            CUDA_TRY(cudaEventRecord(e0));
            if (v == 0) { if ((P == 6 ? pygbe_m2p_launch_6(a) : pygbe_m2p_launch_8(a)) != 0) { pygbe_set_error("mma probe: M2P order %d not built", P); return PYGBE_EINVAL; } }
            else if (v == 1) k_mp_mma<P, 0><<<G, 32, sm0>>>(G, C, d_cell, d_tpos, d_cgeo, d_Bhi, d_Blo, kappa, d_out);
            else if (v == 2) k_mp_mma<P, 1><<<G, 32, sm1>>>(G, C, d_cell, d_tpos, d_cgeo, d_Bhi, d_Blo, kappa, d_out);
            else k_mp_mma<P, 3><<<G, 32, sm3>>>(G, C, d_cell, d_tpos, d_cgeo, d_Bhi, d_Blo, kappa, d_out);
            CUDA_TRY(cudaEventRecord(e1));
            CUDA_TRY(cudaEventSynchronize(e1));
            CUDA_TRY(cudaGetLastError());
            float ms = 0.f;
            CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0) best = std::min(best, ms);
        }
        out[3 * v] = best; out[3 * v + 2] = (double)G * C;
        if (v == 1) { out[3 * v + 1] = NAN; continue; }
        CUDA_TRY(cudaMemcpy(got.data(), d_out, nt * sizeof(double), cudaMemcpyDeviceToHost));
        double en = 0.0;
        for (size_t i = 0; i < nt; i++) en += (got[i] - ref[i]) * (got[i] - ref[i]);
        out[3 * v + 1] = std::sqrt(en / refn);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    for (void *q : {(void *)d_tpos, (void *)d_cgeo, (void *)d_qpos, (void *)d_wc, (void *)d_Bhi, (void *)d_Blo, (void *)d_cell, (void *)d_items, (void *)d_out, (void *)d_ref}) cudaFree(q);
    return PYGBE_OK;
}
