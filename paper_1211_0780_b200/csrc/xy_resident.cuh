// xy_resident.cuh -- the whole Monte Carlo step of SMALL lattices in one persistent kernel (sm_100a):
// SURVEY.md 8(f) f2, stage A (P:30 MCS definition; Eq. 2; Eq. 3).
//
// For L <= 48 a replica's state fits in the shared memory of one SM or of one thread-block cluster.  One
// launch then runs n whole steps -- Metropolis black / white, over-relaxation black / white (+ observables),
// final reduction, replica exchange -- with the spins never leaving the chip:
//
//   * a CTA owns G whole slots (tiny lattices: L = 8 -> 8 slots per CTA), or a cluster of C CTAs owns one
//     slot, each CTA a slab of L/C planes; both colours are resident as fp32 angles AND as (cos, sin) pairs,
//     colour-split like the HBM layout: th_c[slot][zl+1][y][xh], pr_c[...] with one halo plane below and above;
//   * pair == fast_sincos(angle) bit for bit at all times, so a pass never recomputes the (cos, sin) of a
//     neighbour or of a site's own old angle: Metropolis costs 3 MUFU per update (proposal + exp), not 7;
//   * a thread updates the two same-colour sites of one natural quad (one Philox call, R12): both sites are
//     adjacent in the colour-split row, so every neighbour access is one 128-bit shared-memory load;
//   * sites on a slab's first / last plane are also written into the neighbour CTA's halo plane through
//     distributed shared memory (for C = 1 the "neighbour" is the CTA itself: the periodic wrap);
//     one cluster barrier (C > 1) or __syncthreads separates the colour passes;
//   * close Metropolis decisions are settled in fp64 on the spot from the resident angles;
//   * every CTA publishes its fp64 partial sums, the CTAs meet at ONE grid barrier per step (all CTAs are
//     co-resident: cooperative launch), and every CTA then replays the same deterministic exchange
//     decisions, so the beta labels never leave the chip either.
//
// Arithmetic: identical to xy_sweep.cuh site by site (same field summation order, same fast math, same
// Philox keying), so states, permutations and acceptance counts are BITWISE those of the per-pass kernels;
// only the grouping of the fp32 observable terms differs (within the P3 bound).
#pragma once
#include <cooperative_groups.h>
#include "xy_device.cuh"

namespace xyk {
namespace cg = cooperative_groups;

struct ResidentParams {
    float* black; float* white;          // colour-split state in HBM [R][L][L][L/2]
    int R, n_mcs, or_per_mcs;
    int G;                               // slots per CTA (C == 1) or 1
    int tps;                             // threads per slot: a multiple of a plane's items; blockDim.x >= G * tps
    uint32_t n_met0, n_pt0;              // counters of the first step
    PhiloxKeys keys;
    const double* betas;                 // [R] by rank (never changes)
    double* beta_of_slot; float* beta32_of_slot; int* slot_at_rank;     // labels: read at start, written back at the end
    unsigned long long* met_acc; unsigned long long* pt_acc; unsigned long long* exact_count;
    double* obs_rank; double* obs_slot;  // [R][5] of the last step (by rank as measured before its exchange; by slot)
    double* series;                      // [n_mcs][R][5] by rank, or null
    unsigned long long* xchg;            // [2][R][8 CTAs][6] published partial sums E, Mx, My, each as (high half | tag, low half | tag);
                                         // double-buffered by step parity; zero at launch
    unsigned int* sync;                  // [1] error flag (zero at launch)
};

constexpr int kResMaxC = 8;              // portable cluster size
constexpr int kResQueue = 48;            // close decisions a block can defer per colour pass (expected: < 1)
constexpr int kResMaxR = 512;

__host__ __device__ inline size_t resident_smem_bytes(int L, int R, int G, int C) {
    const size_t cs = (size_t)G * (L / C + 2) * L * (L / 2);           // sites of one colour incl. halo planes
    return 2 * cs * 8 + 2 * cs * 4 + 96 * 8 + (size_t)R * (3 * 8 + 3 * 4 + 8) + (size_t)3 * R * C * 8 + (size_t)G * 8 + 64;
}

__device__ __forceinline__ unsigned long long ld_relaxed_gpu(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed_gpu(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// the uniform of exchange pair (k, k+1) of exchange number n_pt (R9, R12, R17)
__device__ __forceinline__ double pt_uniform(int k, uint32_t n_pt, const PhiloxKeys& K) {
    uint32_t w[4];
    philox4x32_10((uint32_t)k, 0u, n_pt, kStreamPT, K, w);
    return (double)w[0] * (1.0 / 4294967296.0);
}

// fp64 definition of one Metropolis decision from resident ANGLES (same formula and neighbour order as
// metropolis_exact / met_fixup_kernel: -x, -y, -z, +x, +y, +z).
__device__ __noinline__ bool metropolis_exact_resident(const float* thO, int ixm, int iym, int izm, int ixp, int iyp, int izp,
                                                       float t_old, float t_new, float u, float beta32) {
    const float nb[6] = { thO[ixm], thO[iym], thO[izm], thO[ixp], thO[iyp], thO[izp] };
    const double lu = accept_log_u((double)u);
    double hx = 0.0, hy = 0.0;
#pragma unroll 1
    for (int j = 0; j < 6; ++j) {
        double s, c;
        sincos_0_2pi((double)nb[j], s, c);
        hx += c; hy += s;
    }
    double so, co, sn, cn;
    sincos_0_2pi((double)t_old, so, co);
    sincos_0_2pi((double)t_new, sn, cn);
    const double dE = -(hx * (cn - co) + hy * (sn - so));
    return accept_exact((double)u, lu, -(double)beta32 * dE);
}

enum { RES_MET = 0, RES_OR = 1, RES_MEAS = 2 };

// Items (quads of one colour) per plane.  The threads of one slot (TPS) are a multiple of it, so that a thread keeps
// ONE (y, xq) for all its planes and its row offsets are computed once; with several slots per block also a multiple
// of 32 (a warp = one slot).  Blocks have at most 512 threads (128 registers each; 1024 threads = 64 registers spill),
// or one plane's items where that is more (L = 48: 576).
__host__ __device__ constexpr int resident_plane_items(int L) { return L * (L / 4); }
__host__ __device__ constexpr int resident_max_threads(int L) {
    return resident_plane_items(L) > 512 ? (resident_plane_items(L) + 31) / 32 * 32 : 512;
}

template <int L, int C>
__global__ void __launch_bounds__(resident_max_threads(L), 1) resident_mcs_kernel(const ResidentParams P) {
    constexpr bool CLUSTER = C > 1;
    constexpr int W = L / 2, XQ = L / 4, PL = L * W, PI = L * XQ;
    constexpr int nz = L / C, SL = (nz + 2) * PL;
    extern __shared__ __align__(16) unsigned char rsm[];
    __shared__ unsigned int s_abort, s_qcount;
    __shared__ uint4 queue[kResQueue];                             // close Metropolis decisions of the current colour pass
    unsigned int* qcount = &s_qcount;

    int crank = 0;
    if (CLUSTER) crank = (int)cg::this_cluster().block_rank();
    const int tid = threadIdx.x, R = P.R;
    const int nS = P.G;
    const int group = blockIdx.x / C;
    const int slot0 = group * nS;
    const int nSloc = min(nS, R - slot0);
    const int z0 = crank * nz;
    const int CS = nS * SL;
    const bool SINGLE = gridDim.x == 1;                            // one CTA holds every slot: no exchange between CTAs

    float2* pr = reinterpret_cast<float2*>(rsm);                 // [2][CS] (cos, sin)
    float* th = reinterpret_cast<float*>(pr + 2 * CS);           // [2][CS] angles
    double* red = reinterpret_cast<double*>(th + 2 * CS);        // [3][32] warp partials
    double* Es = red + 96; double* Mxs = Es + R; double* Mys = Mxs + R;      // by slot, all R
    int* sar = reinterpret_cast<int*>(Mys + R); int* ros = sar + R;          // slot_at_rank, rank_of_slot
    int* sarb = ros + R;                                                      // slot_at_rank before this step's exchange (CTA 0)
    double* betas_s = reinterpret_cast<double*>(sarb + R + (R & 1));          // [R] betas by rank (an even number of ints precedes)
    double* part = betas_s + R;                                               // [3][R*C] collected partial sums (multi-CTA grids)
    float* b32 = reinterpret_cast<float*>(part + (SINGLE ? 0 : 3 * R * C));   // [nS] beta label of the local slots

    // neighbour CTAs' arrays (planes below: rank-1, above: rank+1; periodic).  C == 1: this CTA itself.
    float2 *pr_dn = pr, *pr_up = pr; float *th_dn = th, *th_up = th;
    if (CLUSTER) {
        cg::cluster_group cl = cg::this_cluster();
        pr_dn = cl.map_shared_rank(pr, (crank + C - 1) % C); pr_up = cl.map_shared_rank(pr, (crank + 1) % C);
        th_dn = cl.map_shared_rank(th, (crank + C - 1) % C); th_up = cl.map_shared_rank(th, (crank + 1) % C);
    }
    auto pass_sync = [&]() { if (CLUSTER) cg::this_cluster().sync(); else __syncthreads(); };

    // ---- load: angles of the slab and its two halo planes from HBM, pairs computed once ----------------
    if (tid == 0) { s_abort = 0u; s_qcount = 0u; }
    for (int k = tid; k < R; k += blockDim.x) { const int s = P.slot_at_rank[k]; sar[k] = s; ros[s] = k; betas_s[k] = P.betas[k]; }
    {
        constexpr int W4 = W / 4;                                 // float4 per row
        const int per_col = nSloc * (nz + 2) * L * W4;
        for (int it = tid; it < 2 * per_col; it += blockDim.x) {
            const int c = it >= per_col, j = it - (c ? per_col : 0);
            const int q = j % W4; int r = j / W4;
            const int y = r % L; r /= L;
            const int zp = r % (nz + 2), s = r / (nz + 2);
            int z = z0 + zp - 1; if (z < 0) z += L; if (z >= L) z -= L;
            const float* g = (c ? P.white : P.black) + (size_t)(slot0 + s) * (PL * L) + ((size_t)z * L + y) * W + 4 * q;
            const float4 v = *reinterpret_cast<const float4*>(g);
            const int o = c * CS + s * SL + zp * PL + y * W + 4 * q;
            *reinterpret_cast<float4*>(th + o) = v;
            float sn, cs;
            fast_sincos(v.x, sn, cs); pr[o] = make_float2(cs, sn);
            fast_sincos(v.y, sn, cs); pr[o + 1] = make_float2(cs, sn);
            fast_sincos(v.z, sn, cs); pr[o + 2] = make_float2(cs, sn);
            fast_sincos(v.w, sn, cs); pr[o + 3] = make_float2(cs, sn);
        }
    }
    __syncthreads();
    if (tid < nSloc) b32[tid] = (float)betas_s[ros[slot0 + tid]];
    pass_sync();                                                   // every CTA of the cluster is running and loaded

    // ---- thread -> work: TPS threads per local slot, a thread's items are quads (zl, y, xq) of its slot --
    const int TPS = P.tps;
    const int s = tid / TPS, lt = tid - s * TPS;
    const bool live = s < nSloc;                                   // threads beyond G * TPS (block rounded up to whole warps) idle
    const int slot = slot0 + (live ? s : 0);
    // TPS is a multiple of a plane's items: the thread's (y, xq) is the same on every plane it visits
    const int zl0 = lt / PI, pq = lt - zl0 * PI, PR = TPS / PI;
    const int y = pq / XQ, xq = pq - y * XQ;
    const int oRow = y * W;                                                         // offsets inside a plane (float2 / float units)
    const int oI = oRow + 2 * xq;
    const int oYm = (y == 0 ? L - 1 : y - 1) * W + 2 * xq, oYp = (y + 1 == L ? 0 : y + 1) * W + 2 * xq;
    const int oE0 = oRow + (xq == 0 ? W - 1 : 2 * xq - 1), oE1 = oRow + (2 * xq + 2 == W ? 0 : 2 * xq + 2);   // edge site for par = 0 / 1
    const uint32_t ctrq = (uint32_t)xq + (uint32_t)XQ * (uint32_t)y;               // Philox counter word 0 without the plane
    unsigned int nacc = 0, nexact = 0;
    double dE = 0.0, dMx = 0.0, dMy = 0.0;

    // one colour pass over this CTA's slab; MODE RES_MET / RES_OR / RES_MEAS; accM / accE: add the (new) pairs / the
    // energy terms -S_i.h_i of the own sites to the thread's fp64 sums
    auto pass = [&](const int mode, const int c, const uint32_t n_met, const bool accM, const bool accE) {
        if (!live) return;
        const int o = 1 - c;
        float2* prC = pr + c * CS + s * SL; const float2* prO = pr + o * CS + s * SL;
        float* thC = th + c * CS + s * SL; const float* thO = th + o * CS + s * SL;
        const int offC = c * CS + s * SL;                          // same offsets inside the neighbours' arrays
        float bl = 0.f, win24 = 0.f, beta32 = 0.f;
        if (mode == RES_MET) {
            beta32 = b32[s];
            bl = beta32 * 1.44269504f;
            win24 = (fabsf(beta32) * kWindowPerBeta + kWindowAbs) * 4294967296.0f;
        }
        unsigned int pend = 0u, pend_w = 0u, pend_p = 0u; float pend_old = 0.f;
        for (int zl = zl0; zl < nz; zl += PR) {
            const int z = z0 + zl;
            const int par = (y + z + c) & 1;
            const int pb = (zl + 1) * PL;                          // this plane inside the slot's array
            const int row = pb + oRow, i0 = pb + oI, rym = pb + oYm - 2 * xq, ryp = pb + oYp - 2 * xq;
            const float2 e = prO[pb + (par ? oE1 : oE0)];
            const float4 Cc = *reinterpret_cast<const float4*>(prO + i0);
            const float4 Ym = *reinterpret_cast<const float4*>(prO + rym + 2 * xq), Yp = *reinterpret_cast<const float4*>(prO + ryp + 2 * xq);
            const float4 Zm = *reinterpret_cast<const float4*>(prO + i0 - PL), Zp = *reinterpret_cast<const float4*>(prO + i0 + PL);
            // h = ((S_y- + S_y+) + (S_z- + S_z+)) + (S_x- + S_x+): the summation order of xy_sweep.cuh
            float hx[2], hy[2];
            {
                const float yzAx = (Ym.x + Yp.x) + (Zm.x + Zp.x), yzAy = (Ym.y + Yp.y) + (Zm.y + Zp.y);
                const float yzBx = (Ym.z + Yp.z) + (Zm.z + Zp.z), yzBy = (Ym.w + Yp.w) + (Zm.w + Zp.w);
                const float mx = Cc.x + Cc.z, my = Cc.y + Cc.w;                         // the pair inside the quad
                const float ex = par ? (Cc.z + e.x) : (e.x + Cc.x), ey = par ? (Cc.w + e.y) : (e.y + Cc.y);   // the pair with the edge site
                hx[0] = yzAx + (par ? mx : ex); hy[0] = yzAy + (par ? my : ey);
                hx[1] = yzBx + (par ? ex : mx); hy[1] = yzBy + (par ? ey : my);
            }
            const float2 t2 = *reinterpret_cast<const float2*>(thC + i0);
            float tht[2] = { t2.x, t2.y };
            const float4 own = *reinterpret_cast<const float4*>(prC + i0);
            float pc[2] = { own.x, own.z }, ps[2] = { own.y, own.w };
            bool changed = false;

            if (mode == RES_MET) {
                uint32_t w[4];
                bool closek[2], accf[2]; float told[2];
                philox4x32_10(ctrq + (uint32_t)(XQ * L) * (uint32_t)z, (uint32_t)slot, n_met,
                              c == 0 ? kStreamMetBlack : kStreamMetWhite, P.keys, w);
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const float kf = (float)(w[2 * k] >> 8);
                    const float tn = kf * kTwoPiU24;
                    const float uf = (float)w[2 * k + 1];
                    float sn, cn;
                    fast_sincos(tn, sn, cn);
                    const float g = fmaf(hx[k], cn - pc[k], hy[k] * (sn - ps[k]));       // = -dE; (pc, ps) == fast_sincos(old angle)
                    const float pf = fast_ex2(fmaf(bl, g, 32.0f));
                    const bool acc = uf < pf;
                    closek[k] = fabsf(uf - pf) < win24;            // too close to call in fp32 (no branch here: the two sites' chains interleave)
                    told[k] = tht[k]; accf[k] = acc;
                    if (acc) { tht[k] = tn; pc[k] = cn; ps[k] = sn; ++nacc; changed = true; }
                }
                if (closek[0] | closek[1]) {
                    // rare (4e-5 of the decisions): the fast decision stands for now; the site is remembered in registers,
                    // queued after the loop, and settle_close() re-evaluates it in fp64, eight lanes per site.  A second
                    // close site of the same thread in one pass (probability ~1e-9) is settled on the spot.
#pragma unroll
                    for (int k = 0; k < 2; ++k) {
                        if (!closek[k]) continue;
                        const int xh = 2 * xq + k;
                        const bool fast_acc = accf[k];
                        ++nexact;
                        if (pend == 0u) {
                            pend = 0x40000000u | (unsigned int)zl | ((unsigned int)xh << 8) | ((unsigned int)par << 16) | (fast_acc ? 0x20000u : 0u);
                            pend_old = told[k]; pend_p = w[2 * k]; pend_w = w[2 * k + 1];
                        } else {
                            const int ixm = row + (par ? xh : (xh == 0 ? W - 1 : xh - 1)), ixp = row + (par ? (xh + 1 == W ? 0 : xh + 1) : xh);
                            const float tn = word_to_angle(w[2 * k]);
                            const bool acc = metropolis_exact_resident(thO, ixm, rym + xh, row - PL + xh, ixp, ryp + xh, row + PL + xh,
                                                                       told[k], tn, word_to_u24(w[2 * k + 1]), beta32);
                            if (acc != fast_acc) {
                                tht[k] = acc ? tn : told[k];
                                fast_sincos(tht[k], ps[k], pc[k]);
                                if (acc) ++nacc; else --nacc;
                                changed = true;
                            }
                        }
                    }
                }
            } else if (mode == RES_OR) {
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    float t = fmaf(2.0f, fast_atan2_pos(hy[k], hx[k]), -tht[k]);
                    t = (t < 0.0f) ? t + kTwoPiF : t;
                    t = (t >= kTwoPiF) ? t - kTwoPiF : t;
                    tht[k] = (fmaxf(fabsf(hx[k]), fabsf(hy[k])) > 0.0f) ? t : tht[k];   // R6: h = 0 leaves the spin
                    fast_sincos(tht[k], ps[k], pc[k]);
                }
                changed = true;
            }
            if (accM) { dMx += (double)(pc[0] + pc[1]); dMy += (double)(ps[0] + ps[1]); }
            if (accE) dE -= (double)(fmaf(pc[0], hx[0], ps[0] * hy[0]) + fmaf(pc[1], hx[1], ps[1] * hy[1]));
            if (changed) {
                const float2 ta = make_float2(tht[0], tht[1]);
                const float4 pa = make_float4(pc[0], ps[0], pc[1], ps[1]);
                *reinterpret_cast<float2*>(thC + i0) = ta;
                *reinterpret_cast<float4*>(prC + i0) = pa;
                // halo planes of the neighbours (distributed shared memory; C == 1: the periodic wrap in this CTA)
                if (zl == 0) {
                    const int j = offC + (nz + 1) * PL + y * W + 2 * xq;
                    *reinterpret_cast<float2*>(th_dn + j) = ta; *reinterpret_cast<float4*>(pr_dn + j) = pa;
                }
                if (zl == nz - 1) {
                    const int j = offC + y * W + 2 * xq;
                    *reinterpret_cast<float2*>(th_up + j) = ta; *reinterpret_cast<float4*>(pr_up + j) = pa;
                }
            }
        }
        if (pend) {
            const unsigned int qi = atomicAdd(qcount, 1u);
            const int zl = pend & 0xff, xh = (pend >> 8) & 0xff, par = (pend >> 16) & 1;
            const bool fast_acc = (pend & 0x20000u) != 0u;
            if (qi < kResQueue) {
                queue[qi] = make_uint4((unsigned int)zl | ((unsigned int)y << 8) | ((unsigned int)xh << 16) | ((unsigned int)s << 24) |
                                       ((unsigned int)par << 30) | (fast_acc ? 0x80000000u : 0u), __float_as_uint(pend_old), pend_p, pend_w);
            } else {                                               // queue full (never at ordinary beta): settle on the spot
                const int pb = (zl + 1) * PL, row = pb + oRow;
                const int ixm = row + (par ? xh : (xh == 0 ? W - 1 : xh - 1)), ixp = row + (par ? (xh + 1 == W ? 0 : xh + 1) : xh);
                const float tn = word_to_angle(pend_p);
                const bool acc = metropolis_exact_resident(thO, ixm, pb + oYm - 2 * xq + xh, row - PL + xh, ixp, pb + oYp - 2 * xq + xh, row + PL + xh,
                                                           pend_old, tn, word_to_u24(pend_w), beta32);
                if (acc != fast_acc) {
                    const float tv = acc ? tn : pend_old;
                    float s32, c32;
                    fast_sincos(tv, s32, c32);
                    thC[row + xh] = tv; prC[row + xh] = make_float2(c32, s32);
                    if (zl == 0) { const int j = offC + (nz + 1) * PL + oRow + xh; th_dn[j] = tv; pr_dn[j] = make_float2(c32, s32); }
                    if (zl == nz - 1) { const int j = offC + oRow + xh; th_up[j] = tv; pr_up[j] = make_float2(c32, s32); }
                    if (acc) ++nacc; else --nacc;
                }
            }
        }
    };

    // fp64 settlement of the queued close decisions of colour pass c (after a __syncthreads): the definition of
    // include/xy.h from the resident ANGLES, eight lanes per site like met_fixup_kernel (six neighbours, old angle,
    // proposal: one fp64 sincos each).  Rewrites the site (and its halo copies) with the settled value.
    auto settle_close = [&](const int c) {
        const unsigned int nq = min(*qcount, (unsigned int)kResQueue);
        if (nq == 0u) return;
        const int lane = tid & 31, role = lane & 7, nwarp = blockDim.x >> 5;
        for (unsigned int e0 = (unsigned int)(tid >> 5) * 4u; e0 < nq; e0 += 4u * nwarp) {       // warp-uniform trip count
            const unsigned int e = e0 + (lane >> 3);
            const bool liveq = e < nq;
            const uint4 q = liveq ? queue[e] : make_uint4(0u, 0u, 0u, 0u);
            const int zl = q.x & 0xff, yy = (q.x >> 8) & 0xff, xh = (q.x >> 16) & 0xff, sl = (q.x >> 24) & 0x3f, par = (q.x >> 30) & 1;
            const bool fast_acc = (q.x >> 31) != 0u;
            const float t_old = __uint_as_float(q.y), t_new = word_to_angle(q.z);
            const float* thO = th + (1 - c) * CS + sl * SL;
            const int pb = (zl + 1) * PL, row = pb + yy * W;
            const int rym = pb + (yy == 0 ? L - 1 : yy - 1) * W, ryp = pb + (yy + 1 == L ? 0 : yy + 1) * W;
            int idx = row + xh;
            if (role == 0) idx = row + (par ? xh : (xh == 0 ? W - 1 : xh - 1)); else if (role == 1) idx = rym + xh;
            else if (role == 2) idx = row - PL + xh; else if (role == 3) idx = row + (par ? (xh + 1 == W ? 0 : xh + 1) : xh);
            else if (role == 4) idx = ryp + xh; else if (role == 5) idx = row + PL + xh;
            float a = role == 6 ? t_old : t_new;
            if (role < 6 && liveq) a = thO[idx];
            double sn_, cs_;
            sincos_0_2pi((double)a, sn_, cs_);
            const double uq = (double)word_to_u24(q.w), lu = accept_log_u(uq);          // independent of the fields: overlaps the sincos
            double hx = 0.0, hy = 0.0, co = 0.0, so = 0.0, cn = 0.0, sn = 0.0;
            const int base = lane & ~7;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const double cj = __shfl_sync(0xffffffffu, cs_, base + j), sj = __shfl_sync(0xffffffffu, sn_, base + j);
                if (j < 6) { hx += cj; hy += sj; } else if (j == 6) { co = cj; so = sj; } else { cn = cj; sn = sj; }
            }
            if (liveq && role == 0) {
                const double dEx = -(hx * (cn - co) + hy * (sn - so));
                const bool acc = accept_exact(uq, lu, -(double)b32[sl] * dEx);
                if (acc != fast_acc) {
                    const float tv = acc ? t_new : t_old;
                    float s32, c32;
                    fast_sincos(tv, s32, c32);
                    const int o = c * CS + sl * SL, i = row + xh;
                    th[o + i] = tv; pr[o + i] = make_float2(c32, s32);
                    if (zl == 0) { const int j = o + (nz + 1) * PL + yy * W + xh; th_dn[j] = tv; pr_dn[j] = make_float2(c32, s32); }
                    if (zl == nz - 1) { const int j = o + yy * W + xh; th_up[j] = tv; pr_up[j] = make_float2(c32, s32); }
                    atomicAdd(P.met_acc + slot0 + sl, acc ? 1ull : ~0ull);
                }
            }
        }
        __syncthreads();
        if (tid == 0) *qcount = 0u;
    };

    bool aborted = false;
#ifdef XY_RES_PROF
    long long tk[10]; int nk = 0;
#define RES_TICK() do { if (tid == 0 && blockIdx.x == 0 && t + 1 == P.n_mcs) tk[nk++] = clock64(); } while (0)
#else
#define RES_TICK() do { } while (0)
#endif
    for (int t = 0; t < P.n_mcs && !aborted; ++t) {
        const uint32_t n_met = P.n_met0 + (uint32_t)t, n_pt = P.n_pt0 + (uint32_t)t;
        dE = 0.0; dMx = 0.0; dMy = 0.0;
        // this thread's exchange uniform (pair index = tid), if any, drawn and taken to the log domain HERE, off the
        // critical path: u < exp(x) <=> log(u) < x up to the last bit of either side (far inside P4's 1e-6 window)
        double lu_pt = 0.0;
        if ((int)(n_pt & 1u) + 2 * tid + 1 < R) lu_pt = log(pt_uniform((int)(n_pt & 1u) + 2 * tid, n_pt, P.keys));
        RES_TICK();
        pass(RES_MET, 0, n_met, false, false); __syncthreads(); settle_close(0); pass_sync();
        RES_TICK();
        pass(RES_MET, 1, n_met, false, false); __syncthreads(); settle_close(1); pass_sync();
        RES_TICK();
        for (int j = 0; j < P.or_per_mcs; ++j) {
            const bool last = j + 1 == P.or_per_mcs;
            pass(RES_OR, 0, 0u, last, false); pass_sync();
            pass(RES_OR, 1, 0u, last, last); pass_sync();
        }
        if (P.or_per_mcs == 0) {                                   // no over-relaxation: a reduction pass of its own
            pass(RES_MEAS, 0, 0u, true, false);
            pass(RES_MEAS, 1, 0u, true, true);
        }
        RES_TICK();
        // ---- a4: fixed-order reduction: warp shuffle tree, then the warps of a slot by a second tree (one warp per slot).
        //      Published as self-validating words (half of a double | tag of this step): a reader needs ONE trip to L2 to
        //      see a valid value -- no barrier counter, no fence, no second load.
        const unsigned long long tag = (unsigned long long)(uint32_t)(t + 1);
        unsigned long long* xw = P.xchg + (((size_t)(t & 1) * R + slot) * kResMaxC + crank) * 6;
        {
            double v[3] = { live ? dE : 0.0, live ? dMx : 0.0, live ? dMy : 0.0 };
#pragma unroll
            for (int cidx = 0; cidx < 3; ++cidx)
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) v[cidx] += __shfl_xor_sync(0xffffffffu, v[cidx], off);
            if ((tid & 31) == 0) { red[tid >> 5] = v[0]; red[32 + (tid >> 5)] = v[1]; red[64 + (tid >> 5)] = v[2]; }
            __syncthreads();
            if (lt < 32 && s < nS) {                               // first warp of every slot (a whole warp): lane k holds warp k of the slot
                const int w0 = (s * TPS) >> 5, nw = (TPS + 31) >> 5;
#pragma unroll
                for (int cidx = 0; cidx < 3; ++cidx) {             // the energy first: the exchange waits for it
                    double q = (lt < nw) ? red[32 * cidx + w0 + lt] : 0.0;
#pragma unroll
                    for (int off = 16; off > 0; off >>= 1) q += __shfl_xor_sync(0xffffffffu, q, off);
                    if (lt == 0 && live) {
                        if (SINGLE) (cidx == 0 ? Es : cidx == 1 ? Mxs : Mys)[slot] = q;          // one CTA holds everything
                        else {
                            const unsigned long long qb = (unsigned long long)__double_as_longlong(q);
                            st_relaxed_gpu(xw + 2 * cidx, (qb & 0xffffffff00000000ull) | tag);
                            st_relaxed_gpu(xw + 2 * cidx + 1, (qb << 32) | tag);
                        }
                    }
                }
            }
        }
        RES_TICK();
        if (!SINGLE) {
            // ---- the step's one rendez-vous: every CTA collects the energy of every (slot, slab); CTA 0, which writes the
            //      output rows, also the magnetisation ------------------------------------------------------------------------
            const int nv = blockIdx.x == 0 ? 3 : 1;
            for (int i = tid; i < R * C * nv; i += blockDim.x) {
                const int cidx = i / (R * C), e = i - cidx * (R * C);
                const unsigned long long* x = P.xchg + (((size_t)(t & 1) * R + e / C) * kResMaxC + e % C) * 6 + 2 * cidx;
                unsigned long long a = ld_relaxed_gpu(x), b = ld_relaxed_gpu(x + 1);
                if ((a & 0xffffffffull) != tag || (b & 0xffffffffull) != tag) {
                    const long long t0 = clock64();
                    do {
                        a = ld_relaxed_gpu(x); b = ld_relaxed_gpu(x + 1);
                        if (clock64() - t0 > (1ll << 31)) { s_abort = 1u; atomicExch(P.sync + 1, 1u); break; }   // ~1 s: CTAs not co-resident?
                    } while ((a & 0xffffffffull) != tag || (b & 0xffffffffull) != tag);
                }
                part[i] = __longlong_as_double((long long)((a & 0xffffffff00000000ull) | (b >> 32)));
            }
            __syncthreads();
            if (s_abort) { aborted = true; break; }
            for (int i = tid; i < R * nv; i += blockDim.x) {       // slabs of a slot in fixed order
                const int cidx = i / R, r = i - cidx * R;
                double sum = 0.0;
                for (int k = 0; k < C; ++k) sum += part[cidx * R * C + r * C + k];
                (cidx == 0 ? Es : cidx == 1 ? Mxs : Mys)[r] = sum;
            }
        }
        __syncthreads();
        RES_TICK();
        // ---- a5: every CTA replays the same exchange decisions on its own copy of the labels (the uniforms were drawn
        //      at the top of the step: they do not depend on the energies).  CTA 0 remembers which slot sat at its ranks:
        //      the output rows are those measured BEFORE the exchange (R14) and are written after it, off the other CTAs' path.
        if (blockIdx.x == 0) {
            for (int k = tid; k < R; k += blockDim.x) sarb[k] = sar[k];
            __syncthreads();
        }
        for (int pair = tid, j = 0; ; pair += blockDim.x, ++j) {
            const int k = (int)(n_pt & 1u) + 2 * pair;
            if (k + 1 >= R) break;
            const int a = sar[k], b = sar[k + 1];
            const double lu = j == 0 ? lu_pt : log(pt_uniform(k, n_pt, P.keys));
            if (lu < (betas_s[k] - betas_s[k + 1]) * (Es[a] - Es[b])) {
                sar[k] = b; sar[k + 1] = a; ros[a] = k + 1; ros[b] = k;
                if (blockIdx.x == 0) P.pt_acc[k] += 1ull;
            }
        }
        __syncthreads();
        if (tid < nSloc) b32[tid] = (float)betas_s[ros[slot0 + tid]];
        if (blockIdx.x == 0) {
            const bool last_step = t + 1 == P.n_mcs;
            for (int k = tid; k < R; k += blockDim.x) {
                const int sl = sarb[k];
                const double m2 = Mxs[sl] * Mxs[sl] + Mys[sl] * Mys[sl];
                const double o5[5] = { Es[sl], Mxs[sl], Mys[sl], m2, m2 * m2 };
                for (int cidx = 0; cidx < 5; ++cidx) {
                    if (P.series) P.series[((size_t)t * R + k) * 5 + cidx] = o5[cidx];
                    if (last_step) { P.obs_rank[5 * k + cidx] = o5[cidx]; P.obs_slot[5 * sl + cidx] = o5[cidx]; }
                }
            }
        }
        __syncthreads();
        RES_TICK();
#ifdef XY_RES_PROF
        if (tid == 0 && blockIdx.x == 0 && t + 1 == P.n_mcs)
            printf("resident L=%d C=%d G=%d cycles: metB %lld metW %lld OR %lld reduce+publish %lld collect %lld pt+rows %lld total %lld\n", L, C, nS,
                   tk[1] - tk[0], tk[2] - tk[1], tk[3] - tk[2], tk[4] - tk[3], tk[5] - tk[4], tk[6] - tk[5], tk[6] - tk[0]);
#endif
    }

    // ---- write back: angles of the slab, labels, counters ---------------------------------------------------------------
    {
        constexpr int W4 = W / 4;
        const int per_col = nSloc * nz * L * W4;
        for (int it = tid; it < 2 * per_col; it += blockDim.x) {
            const int c = it >= per_col, j = it - (c ? per_col : 0);
            const int q = j % W4; int r = j / W4;
            const int y = r % L; r /= L;
            const int zl = r % nz, sl = r / nz;
            float* g = (c ? P.white : P.black) + (size_t)(slot0 + sl) * (PL * L) + ((size_t)(z0 + zl) * L + y) * W + 4 * q;
            *reinterpret_cast<float4*>(g) = *reinterpret_cast<const float4*>(th + c * CS + sl * SL + (zl + 1) * PL + y * W + 4 * q);
        }
    }
    if (blockIdx.x == 0)
        for (int k = tid; k < R; k += blockDim.x) {
            const int sl = sar[k];
            P.slot_at_rank[k] = sl; P.beta_of_slot[sl] = P.betas[k]; P.beta32_of_slot[sl] = (float)P.betas[k];
        }
    {
        // widened BEFORE the warp sum: 32 lanes x up to 2^24 steps x the thread's sites does not fit 32 bits (the launcher
        // caps a launch at 2^24 steps, which bounds the per-thread counters themselves)
        unsigned long long a = live ? (unsigned long long)nacc : 0ull, e = live ? (unsigned long long)nexact : 0ull;
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, off); e += __shfl_xor_sync(0xffffffffu, e, off); }
        if ((tid & 31) == 0) {                                     // TPS is a multiple of 32: a warp belongs to one slot
            if (a) atomicAdd(P.met_acc + slot, a);
            if (e) atomicAdd(P.exact_count, e);
        }
    }
    if (CLUSTER) cg::this_cluster().sync();                        // no CTA may leave while a neighbour could still write its halo
}

// by-rank rows from by-slot observables (after the resident kernel: the spins have not moved since)
__global__ void gather_rank_kernel(const double* __restrict__ obs_slot, const int* __restrict__ slot_at_rank, int R,
                                   double* __restrict__ obs_rank) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < 5 * R) obs_rank[i] = obs_slot[5 * slot_at_rank[i / 5] + i % 5];
}

}  // namespace xyk
