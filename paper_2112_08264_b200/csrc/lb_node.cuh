// lb_node.cuh -- the fused one-pass time step with TMA-staged populations, ONE THREAD PER NODE (both components).
//
// Same algorithm, state, shared-memory layout, TMA producer and density ring as lb_tma.cuh (boxes without solid nodes); what
// changes is who does the arithmetic: 8 consumer warps, a thread = a node, holding the 38 populations of BOTH components in
// registers (the producer group hands over its registers: 232 per consumer thread, so nothing spills and no address is recomputed).
// Per node instead of per (node, component): the common velocity u' (S4) is computed once, without the exchange of moments
// and the pair barrier; 1 - 1.5 u'.u', c_i.u' and the symmetric part of the equilibrium at u' are shared by the two components;
// index arithmetic, barrier traffic and loop overhead are paid once.  Fewer warp instructions per node update: at 512^3 the
// step runs at the board's power cap, where instructions cost clock.
#pragma once
#include <cuda.h>

#include "lb_lattice.cuh"
#include "lb_tma.cuh"

namespace lb {

// MODEL 1: the colour-gradient collision (lb_lattice.cuh collide19_cg_pairs, the MODEL 1 variant of k_step_tma)
// instead of Shan-Chen force + BGK.  The recolouring works on the colour-blind sum of the two components, which this thread has
// anyway: one colour-blind collision per node and the two recoloured results, instead of one full collision per component.  The
// ring holds the phase field Theta; G carries sigma.
// DIAG (MODEL 0): the per-component mass and the total momentum of the state after this step, one partial per CTA, as in k_step_tma.
template <typename T, int TY, int MODEL = 0, bool DIAG = false>
__global__ void __launch_bounds__(32 * TY + 128, 1)
k_step_node(const __grid_constant__ CUtensorMap tm_n, const __grid_constant__ CUtensorMap tm_w,
            const __grid_constant__ CUtensorMap tm_c, const T* __restrict__ h, T* __restrict__ g,
            const RhoView<T> ri, const RhoView<T> ro, long long NP, int nx, int ny, int nz, int zc, T om_r, T om_b, T G, int col_split = 1 << 30, T beta = T(0), double* __restrict__ diag_part = nullptr) {
    static_assert(!(MODEL != 0 && DIAG), "the fused sums are built for the Shan-Chen step");
    using L = TmaLayout<T, TY>;
    constexpr int TX = L::TX, NT = L::NT, NC = NT, RW = L::RW, RS = L::RS, SUP = L::SUP, W = L::W, PADX = L::PADX;
    constexpr bool HAS_SOLID = false;
    static_assert(TY >= 2 && TY <= 8, "tile rows");
    // register hand-over between the warp groups: (NT + 128) threads start with 65536 / threads registers each
    constexpr int START_REGS = (65536 / (NC + 128)) / 8 * 8;
    constexpr int PRODUCER_REGS = 32;
    constexpr int CONSUMER_REGS = (START_REGS + (START_REGS - PRODUCER_REGS) * 128 / NC) / 8 * 8;
    extern __shared__ __align__(1024) unsigned char smem_node[];
    unsigned char* smem_tma = smem_node;
    T* sm = reinterpret_cast<T*>(smem_tma);
    T* stage = sm + L::STAGE;
    T* ring = sm + L::RING;
    T* SUb = sm + L::SU;
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_tma + L::BAR_BYTE_OFF);
    unsigned long long* full = bars;          // [2] the 19 boxes of plane `it` have landed in stage it & 1 (tx bytes)
    unsigned long long* done = bars + 2;      // [2] every consumer warp has taken what it needs out of stage it & 1
    unsigned long long* rdy = bars + 4;       // the ring warps have assembled the density ring plane this iteration needs
    unsigned long long* rowpub = bars + 5;    // [2][TY] (of [2][2 TY]) warp ty has published its y-stage inputs of plane `it`

    const int t = threadIdx.x;
    const int ntx = nx / TX, nty = ny / TY;
    const int btx = blockIdx.x, bty = blockIdx.y;
    const int x0 = btx * TX, y0 = bty * TY;
    int z0, niter_cta;
    if (!chunk_range(bty * ntx + btx, col_split, nz, zc, z0, niter_cta)) return;
    // The iteration count differs between CTAs: it lives in shared memory and is re-read where it is used (a register held across
    // the plane loop costs the consumers a spill: +9 local loads per plane, 3.5 % of the step).
    int* const niter_slot = reinterpret_cast<int*>(sm + L::CST + 8);
    auto NITER = [&]() { return *reinterpret_cast<volatile const int*>(niter_slot); };
    auto Z0 = [&]() { return *reinterpret_cast<volatile const int*>(niter_slot + 1); };   // likewise, for the producer group (32 registers)
    const long long pl = (long long)nx * ny;
    const bool wrap_xlo = btx == 0, wrap_xhi = btx == ntx - 1;
    auto wrapz = [&](int p) { p %= nz; return p < 0 ? p + nz : p; };

    if (t == 0) {
        niter_slot[0] = niter_cta; niter_slot[1] = z0;
        sm[L::CST + 5] = T(3) / (T(1) / om_r - T(0.5)); sm[L::CST + 6] = T(3) / (T(1) / om_b - T(0.5));   // 1 / nu_k, nu_k = c_s^2 (tau_k - 1/2)
        for (int s = 0; s < 2; ++s) { mbar_init(full + s, 1); mbar_init(done + s, TY); }
        mbar_init(rdy, 3);
        for (int b = 0; b < 4 * TY; ++b) mbar_init(rowpub + b, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // =================================== producer warp group ===================================
    if (t >= NC) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(PRODUCER_REGS));
        if (t >= NC + 32) {
            // ---- ring warps (3): the density ring, one plane per iteration, two planes ahead of its use.  Ring position
            //      pos (tile + one-node frame) of either component is the sum ((in + x) + y) + xy of up to four single-writer
            //      pieces (lb_onepass.cuh).  Thread r owns positions r, r + 96, ... (at most NPOS = 4) with, for this geometry,
            //      at most one x piece, two y pieces and one xy piece among them: it fetches those pieces itself (cp.async, one
            //      iteration ahead) and only ever reads landing slots it filled itself, so the ring warps need no barrier among
            //      themselves.  Where the pieces live is tabulated once, in shared memory (these warps run on 32 registers):
            //      rt[j][r], j = 0..3 the `in` pieces, 4 the x piece, 5 and 6 the y pieces, 7 the xy piece (element offsets
            //      inside one z plane of their arrays, -1 = none), 8 the positions the extra pieces belong to (2 bits each). ----
            const int r = t - NC - 32;
            constexpr int NR = 96, NPOS = (RS + NR - 1) / NR;
            static_assert(NPOS == 4, "ring table layout");
            int* rt = reinterpret_cast<int*>(sm + L::RTAB) + r;
            {
                int ox = -1, oya = -1, oyb = -1, oxy = -1, who = 0;
#pragma unroll 1
                for (int m = 0; m < NPOS; ++m) {
                    const int pos = r + m * NR;
                    int oin = -1;
                    if (pos < RS) {
                        const int rx = pos % RW - 1, ry = pos / RW - 1;
                        const int txm = btx == 0 ? ntx - 1 : btx - 1, txp = btx == ntx - 1 ? 0 : btx + 1;
                        const int tym = bty == 0 ? nty - 1 : bty - 1, typ = bty == nty - 1 ? 0 : bty + 1;
                        const int otx = rx < 0 ? txm : (rx >= TX ? txp : btx), oty = ry < 0 ? tym : (ry >= TY ? typ : bty);
                        const int lx = rx < 0 ? TX - 1 : (rx >= TX ? 0 : rx), ly = ry < 0 ? TY - 1 : (ry >= TY ? 0 : ry);
                        const bool xe = lx == 0 || lx == TX - 1, ye = ly == 0 || ly == TY - 1;   // edge column / row of its owner tile
                        oin = (oty * TY + ly) * nx + otx * TX + lx;
                        if (xe) {
                            if (ox >= 0) __trap();                         // geometry: one x piece per thread
                            ox = ((oty * ntx + otx) * 2 + (lx != 0)) * TY + ly; who |= m;
                        }
                        if (ye) {
                            const int oy = (oty * 2 + (ly != 0)) * nx + otx * TX + lx;
                            if (oya < 0) { oya = oy; who |= m << 2; }
                            else if (oyb < 0) { oyb = oy; who |= m << 4; }
                            else __trap();                                 // geometry: two y pieces per thread
                        }
                        if (xe && ye) {
                            if (oxy >= 0) __trap();
                            oxy = (oty * ntx + otx) * 4 + (ly != 0) * 2 + (lx != 0); who |= m << 6;
                        }
                    }
                    rt[m * NR] = oin;
                }
                rt[4 * NR] = ox; rt[5 * NR] = oya; rt[6 * NR] = oyb; rt[7 * NR] = oxy; rt[8 * NR] = who;
            }
            const unsigned psx_ = unsigned(nty * ntx * 2 * TY), psy_ = unsigned(nty * 2 * nx), psxy_ = unsigned(nty * ntx * 4);
            T* land = sm + L::LAND + r;                                    // [2][8][96]: per component the 4 `in`, x, y, y, xy landing slots of thread r
            // ask for the pieces of ring plane rp (= box plane z0 - 2 + rp): asynchronous, no registers in flight
            auto ring_fetch = [&](int rp) {
                const unsigned zp = unsigned(wrapz(Z0() - 2 + rp));
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int off = rt[j * NR];
                    if (off >= 0) {
                        const T* b0 = j < 4 ? ri.in : (j == 4 ? ri.x : (j < 7 ? ri.y : ri.xy));
                        const long long cs = j < 4 ? ri.s_in : (j == 4 ? ri.s_x : (j < 7 ? ri.s_y : ri.s_xy));
                        const unsigned ps = j < 4 ? unsigned(pl) : (j == 4 ? psx_ : (j < 7 ? psy_ : psxy_));
                        const T* src = b0 + (zp * ps + unsigned(off));
                        cp_async<sizeof(T)>(land + j * NR, src);
                        cp_async<sizeof(T)>(land + (8 + j) * NR, src + cs);
                    }
                }
                cp_async_commit();
            };
            // ... and add them up in the fixed order ((in + x) + y) + xy once they have landed (own copies only)
            auto ring_assemble = [&](int rp) {
                cp_async_wait<0>();
                T* dst = ring + (rp & 3) * 2 * RS + r;
                const int who = rt[8 * NR];
                const bool hx = rt[4 * NR] >= 0, hya = rt[5 * NR] >= 0, hyb = rt[6 * NR] >= 0, hxy = rt[7 * NR] >= 0;
                const int mx = who & 3, mya = (who >> 2) & 3, myb = (who >> 4) & 3, mxy = (who >> 6) & 3;
#pragma unroll
                for (int kk = 0; kk < 2; ++kk) {
                    const T* ld = land + kk * 8 * NR;
                    T v[NPOS];
#pragma unroll
                    for (int m = 0; m < NPOS; ++m) v[m] = ld[m * NR];
                    const T px = ld[4 * NR], pya = ld[5 * NR], pyb = ld[6 * NR], pxy = ld[7 * NR];
#pragma unroll
                    for (int m = 0; m < NPOS; ++m) {
                        if (hx && mx == m) v[m] += px;
                        if (hya && mya == m) v[m] += pya;
                        if (hyb && myb == m) v[m] += pyb;
                        if (hxy && mxy == m) v[m] += pxy;
                        if (m < NPOS - 1 || r + m * NR < RS) dst[kk * RS + m * NR] = v[m];
                    }
                }
                if (MODEL == 1) {                                           // Theta = (rho^1 - rho^2) / (rho^1 + rho^2), 0 where empty
#pragma unroll
                    for (int m = 0; m < NPOS; ++m)
                        if (m < NPOS - 1 || r + m * NR < RS) {
                            const T a = dst[m * NR], b = dst[RS + m * NR], sum = a + b;
                            dst[m * NR] = sum != T(0) ? (a - b) / sum : T(0);
                        }
                }
            };
            for (int rp = 0; rp < 2; ++rp) {                                // iteration 0 needs ring planes 0, 1, 2
                ring_fetch(rp);
                ring_assemble(rp);
            }
            ring_fetch(2);
            for (int j = 0; j < NITER(); ++j) {
                // ring plane j+2 (the z+1 neighbour plane of iteration j): its slot held plane j-2, last read in iteration
                // j-2, which every consumer warp had left when it arrived on done(j-1)
                if (j > 0) mbar_wait(done + ((j - 1) & 1), ((j - 1) >> 1) & 1);
                ring_assemble(j + 2);
                __syncwarp();
                if ((r & 31) == 0) mbar_arrive(rdy);
                if (j + 3 <= NITER() + 1) ring_fetch(j + 3);
            }
            return;
        }
        // ---- TMA warp: plane j goes into stage j & 1 as soon as every consumer warp has left plane j - 2: a whole iteration
        //      ahead of its use, so the loads come straight from DRAM and need no L2 prefetch ----
        const int lane = t - NC;
        const unsigned long long pol = l2_policy_evict_last();
        for (int j = 0; j < NITER(); ++j) {
            const int z = Z0() - 1 + j;
            const int zw[3] = {wrapz(z - 1), wrapz(z), wrapz(z + 1)};
            if (lane == 0) {
                const int s = j & 1;
                if (j >= 2) mbar_wait(done + s, ((j >> 1) - 1) & 1);
                mbar_expect_tx(full + s, L::STAGE_TX_BYTES + (wrap_xlo ? L::XCOL_TX_BYTES : 0u) + (wrap_xhi ? L::XCOL_TX_BYTES : 0u));
#pragma unroll
                for (int i = 0; i < Q; ++i) {
                    const int zq = zw[1 - dir_cz(i)];                       // f_i(x) = h_i(x - c_i)
                    const int q = pop_plane(0, i);                          // the box takes planes q, q + 1: both components
                    T* slot = stage + s * L::STAGE_ELEMS + L::slot_off(i);
                    if (dir_cx(i) == 0) tma_load_4d(slot, &tm_n, full + s, x0, y0 - dir_cy(i), zq, q, pol);
                    else {
                        tma_load_4d(slot, &tm_w, full + s, dir_cx(i) > 0 ? x0 - PADX : x0, y0 - dir_cy(i), zq, q, pol);
                        // the column beyond the box edge: columns nx-PADX..nx-1 for c_x > 0, 0..PADX-1 for c_x < 0
                        if (dir_cx(i) > 0 && wrap_xlo) tma_load_4d(slot + L::XC, &tm_c, full + s, nx - PADX, y0 - dir_cy(i), zq, q, pol);
                        if (dir_cx(i) < 0 && wrap_xhi) tma_load_4d(slot + L::XC, &tm_c, full + s, 0, y0 - dir_cy(i), zq, q, pol);
                    }
                }
            }
            __syncwarp();
        }
        return;
    }

    // =================================== consumers: one thread per node ===================================
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
    const int tx = t % TX, ty = t / TX;
    const bool lane_lo = tx == 0, lane_hi = tx == TX - 1, row_lo = ty == 0, row_hi = ty == TY - 1;
    const int own_r = (ty + 1) * RW + tx + 1;
    const T zero = T(0);
    const T omc[2] = {T(1) - om_r, T(1) - om_b};
    const unsigned e_own = unsigned((long long)(y0 + ty) * nx + x0 + tx);              // + k NP + z plane stride
    const int btxm = btx == 0 ? ntx - 1 : btx - 1, btxp = btx == ntx - 1 ? 0 : btx + 1;
    const int btym = bty == 0 ? nty - 1 : bty - 1, btyp = bty == nty - 1 ? 0 : bty + 1;
    const unsigned psx = unsigned(nty * ntx * 2 * TY), psy = unsigned(nty * 2 * nx), psxy = unsigned(nty * ntx * 4), plu = unsigned(pl);
    const unsigned step16 = unsigned((NP * (long long)sizeof(T)) >> 4);      // ONE plane: the planes of a direction's two components are adjacent
    const T* ring_n = ring + own_r;                                          // + k RS: density of component k at this node
    T* SUn = SUb + own_r - RW;                                               // + k 2 SUP
    T* exn = sm + L::EX + (ty * 2 + (lane_hi ? 1 : 0)) * 8;                  // + k TY 2 8
    // where this thread finds f_i^k = h_i^k(x - c_i) inside slot i, by c_x (+ the component's offset)
    const int rd0 = ty * TX + tx;
    const int rdp = (wrap_xlo && lane_lo) ? L::XC + ty * PADX + PADX - 1 : ty * W + tx + PADX - 1;
    const int rdm = (wrap_xhi && lane_hi) ? L::XC + ty * PADX : ty * W + tx + 1;
    const int kp = (wrap_xlo && lane_lo) ? TY * PADX : TY * W, km = (wrap_xhi && lane_hi) ? TY * PADX : TY * W;   // component strides of the wide slots
    const bool wrap_ylo = bty == 0 && row_lo, wrap_yhi = bty == nty - 1 && row_hi;
    if (lane_lo || lane_hi) {
#pragma unroll
        for (int k = 0; k < 2; ++k) { exn[k * TY * 16 + 3] = zero; exn[k * TY * 16 + 4] = zero; }
    }
    // z pipelines of the density gather, per component (lb_tma.cuh)
    T qa0[2] = {zero, zero}, qb0[2] = {zero, zero}, qap[2] = {zero, zero}, qbp[2] = {zero, zero}, qam[2] = {zero, zero}, qbm[2] = {zero, zero};
    int zl = wrapz(z0 - 1), zt = wrapz(z0 - 2);

#pragma unroll 1
    for (int it = 0; it < NITER(); ++it) {
        const bool store_h = it >= 1 && it <= NITER() - 2;
        const bool store_rho = it >= 2;
        const int s0 = (it + 1) & 3;
        const int sg = it & 1;
        const unsigned ph = (it >> 1) & 1;
        const T* st = stage + sg * L::STAGE_ELEMS;

        // ---- pull both components: the stage holds h_i^k(x - c_i) for the whole tile (Eq. 5, periodic) ----
        mbar_wait(full + sg, ph);
        mbar_wait(rdy, it & 1);
        T f[2][Q];
#pragma unroll
        for (int k = 0; k < 2; ++k)
#pragma unroll
            for (int i = 0; i < Q; ++i)
                f[k][i] = st[L::slot_off(i) + (dir_cx(i) == 0 ? rd0 + k * NT : (dir_cx(i) > 0 ? rdp + k * kp : rdm + k * km))];
        if (wrap_ylo || wrap_yhi) {                     // the row beyond the box edge in y (one warp of a boundary tile): plain loads
            const int gy = wrap_ylo ? ny - 1 : 0;
            const int x = x0 + tx;
            const int xs[3] = {x == 0 ? nx - 1 : x - 1, x, x == nx - 1 ? 0 : x + 1};
            const long long zs[3] = {(long long)zt * pl, (long long)zl * pl, (long long)(zl + 1 == nz ? 0 : zl + 1) * pl};
#pragma unroll
            for (int k = 0; k < 2; ++k)
#pragma unroll
                for (int i = 1; i < Q; ++i)
                    if (dir_cy(i) != 0) {
                        const T v = __ldg(h + (long long)pop_plane(k, i) * NP + zs[1 - dir_cz(i)] + (long long)gy * nx + xs[1 - dir_cx(i)]);
                        if ((dir_cy(i) > 0 && wrap_ylo) || (dir_cy(i) < 0 && wrap_yhi)) f[k][i] = v;
                    }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");       // generic-proxy reads of the stage before the TMA's next writes
        __syncwarp();
        if (lane_lo) mbar_arrive(done + sg);            // the producer may refill this stage with the plane after next

        T rho[2], jx[2], jy[2], jz[2];
        T ux, uy, uz;
        T ex[2], ey[2], ez[2];
        // MODEL 1: rho[k] the densities, jx[0].. the mixture's momentum, ex[0].. grad Theta, and:
        T cg_rt = zero, cg_x[2] = {zero, zero}, cg_om = zero, cg_amp2 = zero, cg_ig2 = zero, cg_ign = zero, cg_rcs = zero;
        if constexpr (MODEL == 1) {
            // the two densities in the order of moments19, the populations summed over the components
            rho[0] = f[0][0]; rho[1] = f[1][0];
            f[0][0] += f[1][0];
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                rho[0] += f[0][2 * p + 1] + f[0][2 * p + 2];
                rho[1] += f[1][2 * p + 1] + f[1][2 * p + 2];
                f[0][2 * p + 1] += f[1][2 * p + 1]; f[0][2 * p + 2] += f[1][2 * p + 2];
            }
            moments19<T>(f[0], cg_rt, jx[0], jy[0], jz[0]);                // rho and rho u of the mixture (Eq. 7)
            ux = uy = uz = zero;
            ex[0] = ey[0] = ez[0] = zero;
            if (cg_rt != zero) {
                const T irt = T(1) / cg_rt;
                ux = jx[0] * irt; uy = jy[0] * irt; uz = jz[0] * irt;
                cg_x[0] = rho[0] * irt; cg_x[1] = rho[1] * irt;
                const T inv_nu = cg_x[0] * sm[L::CST + 5] + cg_x[1] * sm[L::CST + 6];                 // 1 / nu
                cg_om = T(2) / (T(6) / inv_nu + T(1));                                             // reading C2
                // grad Theta = (1 / c_s^2) sum_i w_i Theta(x + c_i) c_i from the ring (reading C1)
                T d[9];
#pragma unroll
                for (int p = 0; p < 9; ++p) {
                    const int sp = (s0 + pair_cz(p)) & 3, sm_ = (s0 - pair_cz(p)) & 3;
                    d[p] = w_pair<T>(p) * (ring_n[sp * 2 * RS + pair_cy(p) * RW + pair_cx(p)] - ring_n[sm_ * 2 * RS - pair_cy(p) * RW - pair_cx(p)]);
                }
                ex[0] = T(3) * ((((d[0] + d[3]) + d[4]) + d[5]) + d[6]);
                ey[0] = T(3) * ((((d[1] + d[3]) - d[4]) + d[7]) + d[8]);
                ez[0] = T(3) * ((((d[2] + d[5]) - d[6]) + d[7]) - d[8]);
                const T g2 = ex[0] * ex[0] + ey[0] * ey[0] + ez[0] * ez[0];
                if (g2 != zero) { cg_ig2 = T(1) / g2; cg_ign = T(1) / sqrt(g2); }
                cg_amp2 = T(2) * (T(0.5) * (T(2.25) * G * cg_om) * (g2 * cg_ign));                 // 2 (A / 2) |grad|, A = (9/4) sigma omega (Eq. 19)
                cg_rcs = beta * cg_x[0] * cg_x[1] * cg_rt;                                         // beta rho^1 rho^2 / rho (Eq. 20-21)
            }
        } else {
        // ---- moments of both components (Eq. 6-7), common velocity (S4) ----
        moments19<T>(f[0], rho[0], jx[0], jy[0], jz[0]);
        moments19<T>(f[1], rho[1], jx[1], jy[1], jz[1]);
        const T den = om_r * rho[0] + om_b * rho[1];
        const T inv = den != zero ? T(1) / den : zero;
        ux = (om_r * jx[0] + om_b * jx[1]) * inv;
        uy = (om_r * jy[0] + om_b * jy[1]) * inv;
        uz = (om_r * jz[0] + om_b * jz[1]) * inv;
        // ---- du^k = -G sum_i w_i rho^kbar(x+c_i) c_i (S2, S3, S6) from the ring ----
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const T* ro_ = ring_n + (1 - k) * RS;
            T d[9];
#pragma unroll
            for (int p = 0; p < 9; ++p) {
                const int sp = (s0 + pair_cz(p)) & 3, sm_ = (s0 - pair_cz(p)) & 3;
                d[p] = w_pair<T>(p) * (ro_[sp * 2 * RS + pair_cy(p) * RW + pair_cx(p)] - ro_[sm_ * 2 * RS - pair_cy(p) * RW - pair_cx(p)]);
            }
            ex[k] = ux - G * ((((d[0] + d[3]) + d[4]) + d[5]) + d[6]);
            ey[k] = uy - G * ((((d[1] + d[3]) - d[4]) + d[7]) + d[8]);
            ez[k] = uz - G * ((((d[2] + d[5]) - d[6]) + d[7]) - d[8]);
        }

        }
        if constexpr (DIAG) {
            // sum_i f*_i = rho^k and sum_k sum_i f*_i c_i = sum_k (1 - om_k) j^k + rho^k (om_k u' + du^k) (Eq. 1, Eq. 10, S5), which
            // streaming in a periodic box only permutes; the re-collided planes belong to another chunk
            double v0 = 0.0, v1 = 0.0, v2 = 0.0, v3 = 0.0, v4 = 0.0;
            if (store_h) {
                v0 = double(rho[0]); v1 = double(rho[1]);
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const double oc = double(omc[k]), om = 1.0 - oc, r_ = double(rho[k]);
                    v2 += oc * double(jx[k]) + r_ * (om * double(ux) + (double(ex[k]) - double(ux)));
                    v3 += oc * double(jy[k]) + r_ * (om * double(uy) + (double(ey[k]) - double(uy)));
                    v4 += oc * double(jz[k]) + r_ * (om * double(uz) + (double(ez[k]) - double(uz)));
                }
            }
            // four values, 32 lanes: two halving steps, then three plain ones (lanes 0, 8, 16, 24 end up with the sums of v0..v3);
            // the fifth by a plain butterfly
            const bool hA = (tx & 16) != 0, hB = (tx & 8) != 0;
            double kA = hA ? v2 : v0, kB = hA ? v3 : v1;
            kA += __shfl_xor_sync(0xffffffffu, hA ? v0 : v2, 16);
            kB += __shfl_xor_sync(0xffffffffu, hA ? v1 : v3, 16);
            double kk_ = hB ? kB : kA;
            kk_ += __shfl_xor_sync(0xffffffffu, hB ? kA : kB, 8);
            kk_ += __shfl_xor_sync(0xffffffffu, kk_, 4);
            kk_ += __shfl_xor_sync(0xffffffffu, kk_, 2);
            kk_ += __shfl_xor_sync(0xffffffffu, kk_, 1);
#pragma unroll
            for (int o_ = 16; o_ > 0; o_ >>= 1) v4 += __shfl_xor_sync(0xffffffffu, v4, o_);
            double* wacc = reinterpret_cast<double*>(smem_tma + L::WACC_BYTE_OFF) + ty * 8;
            if ((tx & 7) == 0) {
                double* wa = wacc + (hA ? 2 : 0) + (hB ? 1 : 0);
                *wa = (it == 0 ? 0.0 : *wa) + kk_;
            }
            if (tx == 0) wacc[4] = (it == 0 ? 0.0 : wacc[4]) + v4;
        }

        // ---- BGK collision with exact-difference forcing (Eq. 1, Eq. 10, S5) of both components, pair by pair; the stores go out in
        //      plane order (direction-major, the two components adjacent) through one running pointer; the x stage of the density
        //      gather per component as in lb_tma.cuh ----
        T qc0[2] = {zero, zero}, qcp[2] = {zero, zero}, qcm[2] = {zero, zero};
        T* o = g + (e_own + zl * plu);
        auto put = [&](T v) { st_global(o, v); ptr_step16(o, step16); };
        const T a0 = T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz);
        T ae[2] = {zero, zero};
        const T cg_omc = T(1) - cg_om;
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T h0;
            if constexpr (MODEL == 1) {                                    // cos(phi_0) = 0: no recolouring term
                h0 = cg_x[k] * (cg_omc * f[0][0] + cg_om * w_rest<T>() * cg_rt * a0 - cg_amp2 * cg_b_rest<T>());
            } else {
                ae[k] = T(1) - T(1.5) * (ex[k] * ex[k] + ey[k] * ey[k] + ez[k] * ez[k]);
                h0 = omc[k] * f[k][0] + w_rest<T>() * rho[k] * (ae[k] - omc[k] * a0);
            }
            put(h0);
            qb0[k] += h0;
        }
#pragma unroll
        for (int p = 0; p < 9; ++p) {
            const T cu = cdot<T>(p, ux, uy, uz);
            const T s0u = a0 + T(4.5) * cu * cu;
            T h1[2], h2[2];
            if constexpr (MODEL == 1) {                                    // collide19_cg_pairs, once for both components
                const T cg = cdot<T>(p, ex[0], ey[0], ez[0]);
                const T wr = cg_om * (w_pair<T>(p) * cg_rt);
                const T pert = cg_amp2 * (w_pair<T>(p) * cg * cg * cg_ig2 - cg_b_pair<T>(p));             // Eq. 17: the same for i and opp(i)
                const T recol = cg_rcs * w_pair<T>(p) * cg * cg_ign * (p < 3 ? T(1) : T(0.70710678118654752440));   // cos(phi_i)
                const T f1 = cg_omc * f[0][2 * p + 1] + wr * (s0u + T(3) * cu) + pert;
                const T f2 = cg_omc * f[0][2 * p + 2] + wr * (s0u - T(3) * cu) + pert;
                h1[0] = cg_x[0] * f1 + recol; h2[0] = cg_x[0] * f2 - recol;                               // Eq. 20
                h1[1] = cg_x[1] * f1 - recol; h2[1] = cg_x[1] * f2 + recol;                               // Eq. 21
            } else
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const T ce = cdot<T>(p, ex[k], ey[k], ez[k]);
                const T wr = w_pair<T>(p) * rho[k];
                const T se = ae[k] + T(4.5) * ce * ce;
                const T sym = wr * (se - omc[k] * s0u);
                const T asym = (T(3) * wr) * (ce - omc[k] * cu);
                h1[k] = omc[k] * f[k][2 * p + 1] + (sym + asym);
                h2[k] = omc[k] * f[k][2 * p + 2] + (sym - asym);
            }
            put(h1[0]); put(h1[1]); put(h2[0]); put(h2[1]);
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                T* SUup = SUn + k * 2 * SUP + sg * 4 * SUP;
                T* SUum = SUup + SUP;
                T* exs = exn + k * TY * 16;
                T l = zero, r = zero;
                if (p == 0 || (p >= 3 && p <= 6)) { l = __shfl_up_sync(0xffffffffu, h1[k], 1); r = __shfl_down_sync(0xffffffffu, h2[k], 1); }
                if (p == 0) {                                              // +x / -x
                    if (!lane_lo) qb0[k] += l;
                    if (!lane_hi) qb0[k] += r;
                    if (lane_hi) exs[1] = h1[k];
                    if (lane_lo) exs[1] = h2[k];
                } else if (p == 1) { qbp[k] += h1[k]; qbm[k] += h2[k]; }     // +y / -y
                else if (p == 2) { qc0[k] = h1[k]; qa0[k] += h2[k]; }        // +z / -z
                else if (p == 3) {                                         // +x+y / -x-y
                    qbp[k] += lane_lo ? zero : l;
                    qbm[k] += lane_hi ? zero : r;
                    if (lane_hi) SUup[1] = h1[k];
                    if (lane_lo) SUum[-1] = h2[k];
                } else if (p == 4) {                                       // +x-y / -x+y
                    qbm[k] += lane_lo ? zero : l;
                    qbp[k] += lane_hi ? zero : r;
                    if (lane_hi) SUum[1] = h1[k];
                    if (lane_lo) SUup[-1] = h2[k];
                } else if (p == 5) {                                       // +x+z / -x-z
                    if (!lane_lo) qc0[k] += l;
                    if (!lane_hi) qa0[k] += r;
                    if (lane_hi) exs[2] = h1[k];
                    if (lane_lo) exs[0] = h2[k];
                } else if (p == 6) {                                       // +x-z / -x+z
                    if (!lane_lo) qa0[k] += l;
                    if (!lane_hi) qc0[k] += r;
                    if (lane_hi) exs[0] = h1[k];
                    if (lane_lo) exs[2] = h2[k];
                } else if (p == 7) { qcp[k] = h1[k]; qam[k] += h2[k]; }      // +y+z / -y-z
                else { qap[k] += h1[k]; qcm[k] = h2[k]; }                    // +y-z / -y+z
                // corners: only c_z = 0 directions reach a diagonal tile, so the target plane is this plane
                if ((p == 3 || p == 4) && store_h && (lane_lo || lane_hi) && (row_lo || row_hi)) {
                    const bool main_diag = lane_hi == row_hi;
                    if ((p == 3) == main_diag) {
                        const unsigned e_xy = unsigned(k * ro.s_xy) + ((row_hi ? btyp : btym) * ntx + (lane_hi ? btxp : btxm)) * 4 + (row_hi ? (lane_hi ? 0 : 1) : (lane_hi ? 2 : 3));
                        ro.xy[e_xy + zl * psxy] = lane_hi ? h1[k] : h2[k];
                    }
                }
            }
        }
        T p0[2], pp[2], pm[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            p0[k] = qa0[k]; pp[k] = qap[k]; pm[k] = qam[k];                  // complete for plane z-1
            qa0[k] = qb0[k]; qb0[k] = qc0[k];
            qap[k] = qbp[k]; qbp[k] = qcp[k];
            qam[k] = qbm[k]; qbm[k] = qcm[k];
            T* SUup = SUn + k * 2 * SUP + sg * 4 * SUP;
            SUup[0] = pp[k];
            SUup[SUP] = pm[k];
        }
        __syncwarp();
        if (lane_lo) mbar_arrive(rowpub + sg * 2 * TY + ty);

        // ---- the y-edge exports need nothing from the other warps ----
        if ((row_lo || row_hi) && store_rho) {
#pragma unroll
            for (int k = 0; k < 2; ++k) {
                const unsigned e_y = unsigned(k * ro.s_y) + ((row_lo ? btym : btyp) * 2 + (row_lo ? 1 : 0)) * nx + x0 + tx;
                ro.y[e_y + zt * psy] = row_lo ? pm[k] : pp[k];
            }
        }
        {   // the rows above and below have published this plane
            unsigned long long* nb = rowpub + sg * 2 * TY + ty;
            if (row_lo) mbar_wait(nb + 1, ph);
            else if (row_hi) mbar_wait(nb - 1, ph);
            else mbar_wait2(nb - 1, nb + 1, ph);
        }
        // ---- y stage of the gather; exports across the tile's x edges ----
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            T* SUup = SUn + k * 2 * SUP + sg * 4 * SUP;
            T* SUum = SUup + SUP;
            T* exs = exn + k * TY * 16;
            T out = p0[k];
            if (!row_lo) out += SUup[-RW];
            if (!row_hi) out += SUum[RW];
            if (store_rho) ro.in[unsigned(k * NP) + e_own + zt * plu] = out;
            if (lane_lo || lane_hi) {
                const int vc = lane_lo ? -1 : 1;
                T a_0 = exs[1];
                if (!row_lo) a_0 += SUup[vc - RW];
                if (!row_hi) a_0 += SUum[vc + RW];
                const T hout = exs[3] + exs[0];
                exs[3] = exs[4] + a_0;
                exs[4] = exs[2];
                if (store_rho) {
                    const unsigned e_x = unsigned(k * ro.s_x) + ((bty * ntx + (lane_lo ? btxm : btxp)) * 2 + (lane_lo ? 1 : 0)) * TY + ty;
                    ro.x[e_x + zt * psx] = hout;
                }
            }
        }
        zt = zl;
        zl = zl + 1 == nz ? 0 : zl + 1;
    }
    if constexpr (DIAG) {
        asm volatile("bar.sync 9, %0;" ::"n"(NC) : "memory");              // every consumer warp's sums are in place
        if (t < 5) {
            const double* wp = reinterpret_cast<const double*>(smem_tma + L::WACC_BYTE_OFF);
            double s_ = 0.0;
            for (int w_ = 0; w_ < TY; ++w_) s_ += wp[w_ * 8 + t];            // {mass r, mass b, P_x, P_y, P_z}, warps in a fixed order
            const long long cta = blockIdx.x + (long long)gridDim.x * (blockIdx.y + (long long)gridDim.y * blockIdx.z);
            diag_part[cta * 5 + t] = s_;
        }
    }
}

}  // namespace lb
