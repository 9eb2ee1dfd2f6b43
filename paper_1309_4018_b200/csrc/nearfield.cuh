// nearfield.cuh -- direct interactions: P2P (a7), singular / near-singular corrections (a8), density
// weighting and block combination (a9), right-hand side (a10), reaction potential (a12).
#pragma once
#include "common.cuh"
#include "tables.cuh"
#include "blockops.cuh"

// One (target, Gauss point) interaction with the region's kernel, both layers at once (eq. 2 / 9,
// PAPER.md:55-58, :98):   mV G(r) - mK . grad_y G,   G = exp(-kappa r)/r   (1/(4 pi) is in the weights),
//   grad_y G = d (1 + kappa r) exp(-kappa r) / r^3,  d = x - y.
// A pair at zero distance (the K = 4 rule has a node at the collocation point of the self panel,
// reading A5) contributes nothing here; the self panel is handled by the correction (a8).
template <bool YUKAWA>
__device__ __forceinline__ double pair_f64(double dx, double dy, double dz, double mV, double mKx, double mKy,
                                           double mKz, double kappa)
{
    double r2 = dx * dx + dy * dy + dz * dz;
    double rinv = r2 > 0.0 ? rsqrt(r2) : 0.0;
    double mKd = mKx * dx + mKy * dy + mKz * dz;
    double rinv2 = rinv * rinv;
    if (!YUKAWA) {
        return (mV - mKd * rinv2) * rinv;
    } else {
        double kr = kappa * (r2 * rinv);
        double e = exp(-kr);
        return (mV - mKd * (1.0 + kr) * rinv2) * (rinv * e);
    }
}

// ------------------------------------------------------------------------------- per-matvec weighting
// the device slots that VecRef reads (one tiny launch whenever the caller's buffers change)
__global__ void k_set_slots(const double **io, int first, const double *a, const double *b) { io[first] = a; io[first + 1] = b; }

// Gather the densities of the region's panels from x and turn them into point "charges":
//   mV_g = w_g A_j/(4pi) sigma_S c_S dphi_j,   mK_g = w_g A_j/(4pi) sigma_S phi_j n_j     (reading A4)
// and clear the accumulator.
__global__ void k_prep(const int *__restrict__ skip, int np, int K, VecRef xr, const int *__restrict__ phi_idx,
                       const int *__restrict__ dphi_idx, const double *__restrict__ cV,
                       const double *__restrict__ cK, const double4 *__restrict__ pnrm,
                       const double4 *__restrict__ spos, double4 *__restrict__ schg,
                       float4 *__restrict__ schgf, int quad, double *__restrict__ pphi, double *__restrict__ pdphi,
                       double2 *__restrict__ pq, double *__restrict__ out, double *__restrict__ out_twin)
{   // schg: fp64 charges (null in the mixed-precision matvec, whose kernels read schgf only); schgf: fp32 copy,
    // point by point or, with quad = 1, in the quad layout of the packed P2P (p2p.cuh)
    if (skip && *skip) return;
    const long i = blockIdx.x * (long)blockDim.x + threadIdx.x;      // Gauss point
    if (i >= (long)np * K) return;
    const int p = (int)(i / K), g = (int)(i - (long)p * K);
    const double *__restrict__ x = xr.get();
    const double phi = x[phi_idx[p]], dphi = x[dphi_idx[p]];
    const double qV = cV[p] * dphi, qK = cK[p] * phi;
    if (g == 0) {
        pphi[p] = phi; pdphi[p] = dphi;
        if (pq) pq[p] = make_double2(qV, qK);
        out[p] = 0.0;
        if (out_twin) out_twin[p] = 0.0;
    }
    const double4 n = pnrm[p];
    const double w = spos[i].w;
    const double4 c = make_double4(w * qV, w * qK * n.x, w * qK * n.y, w * qK * n.z);
    if (schg) schg[i] = c;
    if (schgf) {
        if (quad) {
            float *f = (float *)schgf + 16 * (i >> 2) + (i & 3);
            f[0] = (float)c.x; f[4] = (float)c.y; f[8] = (float)c.z; f[12] = (float)c.w;
        } else {
            schgf[i] = make_float4((float)c.x, (float)c.y, (float)c.z, (float)c.w);
        }
    }
}

// ------------------------------------------------------------------- singular / near-singular panels
// Step 1: for each target, find the source panels of its group's P2P ranges that are the target's own
// panel or lie inside the near-singular region |x_i - c_j|^2 < thres^2 * 2 A_j  (
// reading A7).  fill == 0 counts, fill == 1 writes column indices (ascending).
// One warp per target: the lanes test 32 consecutive source panels at a time (coalesced), ballots keep the
// column order ascending.
__global__ void __launch_bounds__(128)
k_near_find(int np, const double4 *__restrict__ tpos, const double4 *__restrict__ pnrm,
            const int *__restrict__ p2p_off,
            const int4 *__restrict__ p2p_rng, double thres2, int fill, int *__restrict__ cnt,
            const int *__restrict__ off, int *__restrict__ col)
{
    const int t = (int)((blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (t >= np) return;
    const int g = t / PYGBE_TG;
    const double4 X = tpos[t];
    int n = 0;
    const int base = fill ? off[t] : 0;
    for (int r = p2p_off[g]; r < p2p_off[g + 1]; r++) {
        const int4 rg = p2p_rng[r];
        for (int j0 = rg.x; j0 < rg.y; j0 += 32) {
            const int j = j0 + lane;
            bool near = false;
            if (j < rg.y) {
                const double4 c = tpos[j];
                const double dx = X.x - c.x, dy = X.y - c.y, dz = X.z - c.z;
                near = (j == t) || (thres2 > 0.0 && dx * dx + dy * dy + dz * dz < thres2 * 2.0 * pnrm[j].w);
            }
            const unsigned m = __ballot_sync(0xffffffffu, near);
            if (fill && near) col[base + n + __popc(m & ((1u << lane) - 1u))] = j;
            n += __popc(m);
        }
    }
    if (!fill && lane == 0) cnt[t] = n;
}

// Semi-analytic self integral of the single-layer kernel (PAPER.md:165 [22], :235 "N_k"; reading A6):
// polar coordinates about the centroid in the panel plane, radial integral analytic
//   int_0^R exp(-kappa r) dr = R  or  (1 - exp(-kappa R))/kappa,   R(theta) = h / cos(theta),
// angular integral by N_k-point Gauss-Legendre on each side's angular interval.  Without 1/(4 pi).
__device__ double self_integral(const double *t, double kappa, const QuadTables &q)
{
    double c[3] = {(t[0] + t[3] + t[6]) / 3.0, (t[1] + t[4] + t[7]) / 3.0, (t[2] + t[5] + t[8]) / 3.0};
    double total = 0.0;
    for (int s = 0; s < 3; s++) {
        const double *a = t + 3 * s, *b = t + 3 * ((s + 1) % 3);
        double e[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]};
        double len = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2]);
        e[0] /= len; e[1] /= len; e[2] /= len;
        double ac[3] = {a[0] - c[0], a[1] - c[1], a[2] - c[2]};
        double sa = ac[0] * e[0] + ac[1] * e[1] + ac[2] * e[2];
        double sb = sa + len;
        double px = ac[0] - sa * e[0], py = ac[1] - sa * e[1], pz = ac[2] - sa * e[2];
        double h = sqrt(px * px + py * py + pz * pz);
        double th1 = atan2(sa, h), th2 = atan2(sb, h);
        double half = 0.5 * (th2 - th1), mid = 0.5 * (th2 + th1), acc = 0.0;
        for (int k = 0; k < q.Nk; k++) {
            double R = h / cos(mid + half * q.glx[k]);
            acc += q.glw[k] * (kappa == 0.0 ? R : (1.0 - exp(-kappa * R)) / kappa);
        }
        total += half * acc;
    }
    return total;
}

// Step 2: value of each correction entry = (fine rule or semi-analytic) - (what P2P adds with the K-point
// rule), for the single- and the double-layer kernel, with sigma_S c_S / sigma_S of the source panel
// folded in.  One warp per target row, lanes over its entries.  Self panel: V = semi-analytic, K = 0 (flat panel).
__global__ void k_near_values(int np, QuadTables q, bool yukawa, double kappa, const int *__restrict__ off,
                              const int *__restrict__ col, const int *__restrict__ gid,
                              const double *__restrict__ tri, const double4 *__restrict__ tpos,
                              const double4 *__restrict__ pnrm, const double4 *__restrict__ spos,
                              const double *__restrict__ cV, const double *__restrict__ cK,
                              double2 *__restrict__ val)
{
    const int t = (int)((blockIdx.x * (long)blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (t >= np) return;
    double4 X = tpos[t];
    const double inv4pi = 0.07957747154594767;
    for (int e = off[t] + lane; e < off[t + 1]; e += 32) {
        int j = col[e];
        double4 nA = pnrm[j];
        // coarse part, exactly as k_p2p evaluates it (unit densities)
        double cv = 0.0, ck = 0.0;
        for (int g = 0; g < q.K; g++) {
            double4 a = spos[(long)j * q.K + g];
            double dx = X.x - a.x, dy = X.y - a.y, dz = X.z - a.z;
            if (yukawa) {
                cv += pair_f64<true>(dx, dy, dz, a.w, 0, 0, 0, kappa);
                ck -= pair_f64<true>(dx, dy, dz, 0, a.w * nA.x, a.w * nA.y, a.w * nA.z, kappa);
            } else {
                cv += pair_f64<false>(dx, dy, dz, a.w, 0, 0, 0, kappa);
                ck -= pair_f64<false>(dx, dy, dz, 0, a.w * nA.x, a.w * nA.y, a.w * nA.z, kappa);
            }
        }
        const double *tj = tri + 9 * (long)gid[j];
        double fv = 0.0, fk = 0.0;
        if (j == t) {
            fv = self_integral(tj, kappa, q) * inv4pi;
            fk = 0.0;
        } else {
            for (int g = 0; g < q.Kfine; g++) {
                double b0 = q.bF[g][0], b1 = q.bF[g][1], b2 = q.bF[g][2];
                double yx = b0 * tj[0] + b1 * tj[3] + b2 * tj[6];
                double yy = b0 * tj[1] + b1 * tj[4] + b2 * tj[7];
                double yz = b0 * tj[2] + b1 * tj[5] + b2 * tj[8];
                double w = q.wF[g] * nA.w * inv4pi;
                double dx = X.x - yx, dy = X.y - yy, dz = X.z - yz;
                if (yukawa) {
                    fv += pair_f64<true>(dx, dy, dz, w, 0, 0, 0, kappa);
                    fk -= pair_f64<true>(dx, dy, dz, 0, w * nA.x, w * nA.y, w * nA.z, kappa);
                } else {
                    fv += pair_f64<false>(dx, dy, dz, w, 0, 0, 0, kappa);
                    fk -= pair_f64<false>(dx, dy, dz, 0, w * nA.x, w * nA.y, w * nA.z, kappa);
                }
            }
        }
        val[e] = make_double2(cV[j] * (fv - cv), cK[j] * (fk - ck));
    }
}

// Correction SpMV (a8) for a region and, optionally, its twin (same sparsity pattern, own values):
//   corr[t] = sum_e [ val.x dphi_j - val.y phi_j ].
// It needs only the gathered densities, so it runs on its own stream beside the P2P / M2P and is
// latency-bound (~50 entries per row): four lanes share a row, partial sums meet by shuffles in a fixed order.
#define NEAR_LANES 4
__global__ void __launch_bounds__(128)
k_near(const int *__restrict__ skip, int np, const int *__restrict__ off, const int *__restrict__ col,
       const double2 *__restrict__ valA, const double2 *__restrict__ valB, const double *__restrict__ pphi,
       const double *__restrict__ pdphi, double *__restrict__ corrA, double *__restrict__ corrB)
{
    if (skip && *skip) return;
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int t = gt / NEAR_LANES, lane = gt % NEAR_LANES;
    double accA = 0.0, accB = 0.0;
    if (t < np) {
        const int e0 = off[t], e1 = off[t + 1];
        if (valB) {
#pragma unroll 2
            for (int e = e0 + lane; e < e1; e += NEAR_LANES) {
                const int j = col[e];
                const double ph = pphi[j], dp = pdphi[j];
                const double2 a = valA[e], b = valB[e];
                accA += a.x * dp - a.y * ph;
                accB += b.x * dp - b.y * ph;
            }
        } else {
#pragma unroll 2
            for (int e = e0 + lane; e < e1; e += NEAR_LANES) {
                const int j = col[e];
                const double2 a = valA[e];
                accA += a.x * pdphi[j] - a.y * pphi[j];
            }
        }
    }
#pragma unroll
    for (int o = 1; o < NEAR_LANES; o <<= 1) {
        accA += __shfl_xor_sync(0xffffffffu, accA, o);
        accB += __shfl_xor_sync(0xffffffffu, accB, o);
    }
    if (t < np && lane == 0) { corrA[t] = accA; if (valB) corrB[t] = accB; }
}

// Block combination (a9), eq. (10):  y[row] = 1/2 phi - ( out + corr ).
__global__ void k_combine(const int *__restrict__ skip, int np, const double *__restrict__ pphi,
                          const double *__restrict__ outA, const double *__restrict__ outB,
                          const double *__restrict__ corrA, const double *__restrict__ corrB,
                          const int *__restrict__ rowA, const int *__restrict__ rowB, VecRef yr)
{
    if (skip && *skip) return;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= np) return;
    double *__restrict__ y = const_cast<double *>(yr.get());
    const double half_phi = 0.5 * pphi[t];
    y[rowA[t]] = half_phi - (outA[t] + corrA[t]);
    if (outB) y[rowB[t]] = half_phi - (outB[t] + corrB[t]);
}

// ------------------------------------------------------------------------------------------------ RHS
// b[row(Omega,T,i)] = sum_{k in Omega} q_k G_Omega(x_i, r_k) / eps_Omega   (eq. 9 / 11).
#define RHS_TILE 256
template <bool YUKAWA>
__global__ void __launch_bounds__(128)
k_rhs(int np, const double4 *__restrict__ tpos, const int *__restrict__ row_idx, int nq,
      const double4 *__restrict__ qpos, double kappa, double inv_eps_4pi, double *__restrict__ b)
{
    __shared__ double4 s_q[RHS_TILE];
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    bool ok = t < np;
    double4 X = ok ? tpos[t] : make_double4(0, 0, 0, 0);
    double acc = 0.0;
    for (int base = 0; base < nq; base += RHS_TILE) {
        int n = min(RHS_TILE, nq - base);
        __syncthreads();
        for (int i = threadIdx.x; i < n; i += blockDim.x) s_q[i] = qpos[base + i];
        __syncthreads();
        for (int i = 0; i < n; i++) {
            double4 a = s_q[i];
            acc += pair_f64<YUKAWA>(X.x - a.x, X.y - a.y, X.z - a.z, a.w, 0, 0, 0, kappa);
        }
    }
    if (ok) b[row_idx[t]] = acc * inv_eps_4pi;
}

// ------------------------------------------------------------------------------- reaction potential
// phi_reac(r_k) = sum_{S in dOmega} sigma_S [ c_S V dphi_S - K phi_S ](r_k)  with the plain K-point rule
// (eq. 4; discretised :119).  The point charges schg come from k_prep with the solution.
// grid = (charges, source chunks): the charges are on grid.x, which has no practical limit (a region may hold
// more than the 65535 that grid.y allows); block reduce, one atomicAdd per CTA.
#define EN_THREADS 256
#define EN_CHUNK 4096
template <bool YUKAWA>
__global__ void __launch_bounds__(EN_THREADS)
k_reaction(int npts, const double4 *__restrict__ spos, const double4 *__restrict__ schg, int nq,
           const double4 *__restrict__ qpos, const int *__restrict__ qid, double kappa,
           double *__restrict__ phi_reac)
{
    int k = blockIdx.x;
    double4 X = qpos[k];
    long lo = (long)blockIdx.y * EN_CHUNK, hi = min((long)npts, lo + EN_CHUNK);
    double acc = 0.0;
    for (long i = lo + threadIdx.x; i < hi; i += EN_THREADS) {
        double4 a = spos[i], c = schg[i];
        acc += pair_f64<YUKAWA>(X.x - a.x, X.y - a.y, X.z - a.z, c.x, c.y, c.z, c.w, kappa);
    }
    double s = block_sum<EN_THREADS>(acc);
    if (threadIdx.x == 0) atomicAdd(phi_reac + qid[k], s);
}

// sum_k q_k phi_reac[k] (eq. 6) -> out[0]; single CTA.
__global__ void __launch_bounds__(256) k_dot_q(int nq, const double *__restrict__ q,
                                               const double *__restrict__ phi, double *__restrict__ out)
{
    double acc = 0.0;
    for (int i = threadIdx.x; i < nq; i += 256) acc += q[i] * phi[i];
    double s = block_sum<256>(acc);
    if (threadIdx.x == 0) out[0] = s;
}

// Coulomb energy sum over pairs inside one region (eq. 8): sum_{k != l} q_k q_l / r_kl.
__global__ void __launch_bounds__(128) k_coulomb(int nq, const double4 *__restrict__ qpos, double *__restrict__ out)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    double acc = 0.0;
    if (k < nq) {
        double4 X = qpos[k];
        for (int l = 0; l < nq; l++) {
            double4 a = qpos[l];
            acc += pair_f64<false>(X.x - a.x, X.y - a.y, X.z - a.z, a.w, 0, 0, 0, 0.0);   // r = 0 -> 0
        }
        acc *= X.w;
    }
    double s = block_sum<128>(acc);
    if (threadIdx.x == 0) atomicAdd(out, s);
}
