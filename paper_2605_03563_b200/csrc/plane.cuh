// plane.cuh — the plane-pipeline stencil engine (2.5-D blocking).  One template serves every pass whose core is
// "form a vector v point by point, take out = L_h v, then a pointwise epilogue with fused dot products":
// stencil apply / residual, the CG pass {p-update + matvec + p.Ap} and the two BiCGSTAB matvec
// passes.
//
// Geometry: a CTA owns an xy tile of TX x TY = 128 x 16 points and marches a chunk of z planes.  Threads are
// 64 x 8; each owns two x-adjacent points (one 16-byte access) in two adjacent rows.  The formed vector v lives in
// a shared-memory ring of 2R+2 planes, each (TY+2R) x (TX+2HX) with its xy halo (R = stencil radius, HX = halo
// rounded up to whole 16-byte pairs), so v is formed ONCE per point per pass (halo points once more by the
// neighbouring CTA) and all 6R neighbours of a point come from shared memory.  Loads for plane k+R+1 are issued a
// full iteration before they are consumed (software pipelining through registers), one __syncthreads per plane.
// Out-of-range neighbours follow include/poisson.h: periodic wrap, ghost-face values, or zero.
// Arithmetic order is the canonical one of stencil.cuh, so results are bit-identical to the generic kernels.
#pragma once
#include <algorithm>
#include <cstdlib>

#include "stencil.cuh"

namespace pb {

__device__ __forceinline__ double2 ld2(const double* p) { return *reinterpret_cast<const double2*>(p); }
__device__ __forceinline__ void st2(double* p, double2 v) { *reinterpret_cast<double2*>(p) = v; }
__device__ __forceinline__ double2 mk2(double a, double b) { return make_double2(a, b); }

// Tile configuration: TX x TY points per CTA, RPT rows per thread (threads = TX/2 x TY/RPT), MINB resident CTAs per
// SM asked of the compiler, PF = how many planes ahead the global loads run.
template <int TX_, int TY_, int RPT_, int MINB_, int PF_, int ZQ_ = 0, int YW_ = 1>
struct TileCfg {
    static constexpr int TX = TX_, TY = TY_, RPT = RPT_, MINB = MINB_, PF = PF_;
    static constexpr int YW = YW_;  // radius 3: read the y window of all owned rows once per plane (else per row)
    static constexpr int ZQ = ZQ_;  // radius 3 only: keep the z neighbours of the owned points in a register queue
};

template <int KIND, class Cfg>
struct PlaneGeom {
    static constexpr int R = (KIND == KIND_CART6) ? 3 : 1;
    static constexpr int HX = (R == 1) ? 2 : 4;
    static constexpr int TX = Cfg::TX, TY = Cfg::TY, RPT = Cfg::RPT, PF = Cfg::PF;
    static constexpr int NTX = TX / 2, NTY = TY / RPT, NT = NTX * NTY;
    static constexpr int SW = TX + 2 * HX, SH = TY + 2 * R;
    static constexpr int NS = 2 * R + 2;  // power of two (4 or 8)
    static constexpr int SLOT = SH * SW;
    static constexpr size_t SMEM = (size_t)NS * SLOT * sizeof(double);
    static constexpr int NHALO = R * TX + TY * HX;        // halo pairs per plane: 2R rows x TX/2 + TY rows x HX
    static constexpr int NH = (NHALO + NT - 1) / NT;      // halo pairs per thread
};

// Value of the loader's vector at (i,j,k) when at most one index is out of range (slow path: boundary cells only).
// Edge and corner ghosts are never read by a star stencil and come back as zero.
template <class Ld>
__device__ double vpoint(const Op& op, const Ld& ld, int i, int j, int k, bool ug) {
    int id[3] = {i, j, k};
    int bad = -1, nbad = 0;
#pragma unroll
    for (int a = 0; a < 3; ++a)
        if (id[a] < 0 || id[a] >= op.n[a]) {
            bad = a;
            ++nbad;
        }
    if (nbad == 0) return ld.at(op, gidx(op, i, j, k), i, j, k);
    if (nbad > 1) return 0.0;
    const int n = op.n[bad], q = id[bad];
    const int f = 2 * bad + (q < 0 ? 0 : 1), bc = op.bc[f];
    if (bc == POISSON_BC_PERIODIC) {
        id[bad] = ((q % n) + n) % n;
        return ld.at(op, gidx(op, id[0], id[1], id[2]), id[0], id[1], id[2]);
    }
    if (bc == POISSON_BC_DIRICHLET_GHOST && ug && op.ghost[f] != nullptr) {
        const int layer = q < 0 ? (-1 - q) : (q - n);
        if (layer >= op.R) return 0.0;
        const int a1 = (bad == 0) ? 1 : 0, a2 = (bad == 2) ? 1 : 2;
        return op.ghost[f][((size_t)layer * op.n[a2] + id[a2]) * op.n[a1] + id[a1]];
    }
    return 0.0;
}

// Per-thread coefficients of the operator rows it owns.
template <int KIND, int RPT>
struct RowCoef {};
template <int RPT>
struct RowCoef<KIND_CART2, RPT> {
    double c0, c1, c2, d;
    bool plain;
};
template <int RPT>
struct RowCoef<KIND_CART6, RPT> {
    double c0, c1, c2, d;
};
template <int RPT>
struct RowCoef<KIND_SPH, RPT> {
    double arm[2], arp[2], ir2[2], dr[2];          // per own column
    double atm[RPT], atp[RPT], cp[RPT], dt[RPT];   // per own row
};

// Loader / epilogue concepts (see k_plane.cu for the instances):
//   struct Ld { struct Raw; static bool PLAIN, SIDE, USES_DIAG (then: double2 form_own(const Raw&, double d0, double d1)); void prepare(); Raw load(size_t p) const; Raw load_own(size_t p) const;
//               void side(const Raw&, size_t p) const;   (pointwise side effect on owned points, e.g. the CG x-update)
//               double2 form(const Op&, const Raw&, int i, int j, int k) const;   (pair starting at column i)
//               double at(const Op&, size_t p, int i, int j, int k) const; };
//   struct Ep { static constexpr int NRED; struct Raw; bool skip() const; void prepare(); Raw load(size_t p) const;
//               void apply(const Raw&, size_t p, int i, int j, int k, double2 v, double2 lv, double* acc) const;
//               void finish(const double* totals) const; };
template <int KIND, class Cfg, class Ld, class Ep>
__global__ void __launch_bounds__(PlaneGeom<KIND, Cfg>::NT, Cfg::MINB)
    k_plane(const Op op, const Ld ld_in, const Ep ep_in, const long items, const int per_tile, const int ntx, const bool ug_in,
            RedBuf rb) {
    using G = PlaneGeom<KIND, Cfg>;
    constexpr int R = G::R, HX = G::HX, TX = G::TX, TY = G::TY, SW = G::SW, NS = G::NS, SLOT = G::SLOT;
    constexpr int RPT = G::RPT, NH = G::NH, PF = G::PF;
    extern __shared__ __align__(16) double ring[];
    if (ep_in.skip()) return;
    Ld ld = ld_in;  // the functors fetch their device-resident scalars (alpha, beta, ...) once
    Ep ep = ep_in;
    ld.prepare();
    ep.prepare();
    const bool ug = ug_in && op.gamma == 0.0;
    const int n0 = op.n[0], n1 = op.n[1], n2 = op.n[2];
    const int lx = threadIdx.x, ty = threadIdx.y, tid = ty * G::NTX + lx;
    double acc[Ep::NRED > 0 ? Ep::NRED : 1];
#pragma unroll
    for (int r = 0; r < (Ep::NRED > 0 ? Ep::NRED : 1); ++r) acc[r] = 0.0;
    // Work = (tile, plane) items; every CTA takes one contiguous run of them, cut into (tile, k0..k1) segments.
    const long total = (long)ntx * ((n1 + TY - 1) / TY) * n2;
    // per_tile > 0: whole z chunks, per_tile runs per tile (a run never straddles two tiles); else one linear split
    long pos = (long)blockIdx.x * items;
    long pend = min(total, pos + items);
    if (per_tile > 0) {
        const long t0 = (long)(blockIdx.x / per_tile) * n2;
        pos = t0 + (long)(blockIdx.x % per_tile) * items;
        pend = min(t0 + n2, pos + items);
    }
    while (pos < pend) {
    const int tile = (int)(pos / n2), k0 = (int)(pos % n2);
    const int k1 = (int)min((long)n2, (long)k0 + (pend - pos));
    pos += k1 - k0;
    const int i0 = (tile % ntx) * TX, j0 = (tile / ntx) * TY;
    __syncthreads();  // the previous segment's readers are done with the ring
    const int i = i0 + 2 * lx;
    const int jrow = j0 + RPT * ty;  // first owned row
    bool act[RPT];
#pragma unroll
    for (int r = 0; r < RPT; ++r) act[r] = i < n0 && jrow + r < n1;
    const size_t plane = (size_t)n0 * n1;
    const size_t base0 = (size_t)jrow * n0 + i;               // row r: base0 + r*n0
    const int so0 = (R + RPT * ty) * SW + HX + 2 * lx;        // row r: so0 + r*SW
    const bool per_z = op.bc[4] == POISSON_BC_PERIODIC;

    // ---- this thread's halo pairs ----------------------------------------------------------------------------------
    // class 0 none, 1 plain load at the wrapped (hwi,hwj), 2 boundary values through vpoint()
    int hcls[NH], hi[NH], hj[NH], hso[NH], hwi[NH], hwj[NH];
#pragma unroll
    for (int m = 0; m < NH; ++m) {
        const int h = tid + m * G::NT;
        hcls[m] = 0;
        hi[m] = hj[m] = hso[m] = hwi[m] = hwj[m] = 0;
        if (h < R * TX) {  // rows above and below the tile
            const int rr = h / G::NTX, c = h % G::NTX;
            const int srow = rr < R ? rr : TY + rr;
            hj[m] = j0 - R + srow;
            hi[m] = i0 + 2 * c;
            hso[m] = srow * SW + HX + 2 * c;
            hcls[m] = 1;
        } else if (h < G::NHALO) {  // columns left and right of the tile
            const int t = h - R * TX, row = t / HX, c = t % HX;
            const int pc = c < HX / 2 ? c : (TX / 2 + c);
            hj[m] = j0 + row;
            hi[m] = i0 - HX + 2 * pc;
            hso[m] = (R + row) * SW + 2 * pc;
            hcls[m] = 1;
        }
        if (hcls[m]) {
            const bool ox = hi[m] < 0 || hi[m] >= n0, oy = hj[m] < 0 || hj[m] >= n1;
            hwi[m] = hi[m];
            hwj[m] = hj[m];
            if (ox && oy) {
                hcls[m] = 0;
            } else if (ox) {
                if (op.bc[0] == POISSON_BC_PERIODIC && n0 >= HX) hwi[m] = ((hi[m] % n0) + n0) % n0; else hcls[m] = 2;
            } else if (oy) {
                if (op.bc[2] == POISSON_BC_PERIODIC) hwj[m] = ((hj[m] % n1) + n1) % n1; else hcls[m] = 2;
            }
        }
    }

    // ---- operator coefficients of the owned rows ----------------------------------------------------------------
    RowCoef<KIND, RPT> rc;
    if constexpr (KIND == KIND_SPH) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            const int ii = min(i + e, n0 - 1);
            rc.arm[e] = op.ar_m[ii];
            rc.arp[e] = op.ar_p[ii];
            rc.ir2[e] = op.ir2[ii];
            rc.dr[e] = op.dr[ii];
        }
#pragma unroll
        for (int r = 0; r < RPT; ++r) {
            const int jj = min(jrow + r, n1 - 1);
            rc.atm[r] = op.at_m[jj];
            rc.atp[r] = op.at_p[jj];
            rc.cp[r] = op.cp[jj];
            rc.dt[r] = op.dt[jj];
        }
    } else {
        rc.c0 = op.c[0];
        rc.c1 = op.c[1];
        rc.c2 = op.c[2];
        if constexpr (KIND == KIND_CART6) {
            rc.d = (49.0 / 18.0) * ((rc.c0 + rc.c1) + rc.c2);
        } else {
            rc.d = 2.0 * ((rc.c0 + rc.c1) + rc.c2);
            bool neumann = false;
#pragma unroll
            for (int f = 0; f < 6; ++f) neumann |= op.bc[f] == POISSON_BC_NEUMANN0;
            rc.plain = !neumann && op.gamma == 0.0;
        }
    }

    // diagonals of this thread's halo points (spherical operator: fixed along the marching axis)
    double hd0[NH], hd1[NH];
#pragma unroll
    for (int m = 0; m < NH; ++m) {
        hd0[m] = hd1[m] = 1.0;
        if constexpr (KIND == KIND_SPH) {
            if (hcls[m] == 1) {
                hd0[m] = row_diag<double, KIND_SPH>(op, hwi[m], hwj[m], 0);
                hd1[m] = row_diag<double, KIND_SPH>(op, min(hwi[m] + 1, n0 - 1), hwj[m], 0);
            }
        }
    }

    // spherical operator + a loader that divides by the diagonal and asks for it (Ld::RECIP; it pays where registers
    // allow: BiCGSTAB pass 2 86 -> 80 us, pass 1 97 -> 104 us): divisor and reciprocal once per column, not per plane
    constexpr bool sph_rd = KIND == KIND_SPH && [] { if constexpr (requires { Ld::RECIP; }) return Ld::USES_DIAG && Ld::RECIP; else return false; }();
    double odv[RPT][2], ord_[RPT][2];
    if constexpr (sph_rd) {
#pragma unroll
        for (int r = 0; r < RPT; ++r)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                odv[r][e] = ld.divisor(fma(rc.ir2[e], rc.dt[r], rc.dr[e]));
                ord_[r][e] = 1.0 / odv[r][e];
            }
#pragma unroll
        for (int m = 0; m < NH; ++m) {  // hd0 / hd1 become divisor, and two more registers hold the reciprocals
            hd0[m] = ld.divisor(hd0[m]);
            hd1[m] = ld.divisor(hd1[m]);
        }
    }

    // ---- plane staging --------------------------------------------------------------------------------------------
    struct Staged {
        typename Ld::Raw o[RPT], h[NH];
        int kw;       // wrapped plane index, or -1 when the plane lies outside a non-periodic z face
    };
    constexpr bool ZQ = (KIND == KIND_CART6) && (Cfg::ZQ != 0);
    double2 zq[ZQ ? RPT : 1][2 * R + 1];
    // Boundary values (ghost faces, zeros, wrapped tiny grids) come through vpoint().  For a PLAIN loader (the vector is
    // an array: Raw is the pair itself) they are fetched here, with the plane's other loads, so that their latency is
    // hidden like any other; the Krylov loaders never see ghost values and resolve them at commit time.
    auto bpair = [&](int ii, int jj, int kk) { return mk2(vpoint(op, ld, ii, jj, kk, ug), vpoint(op, ld, ii + 1, jj, kk, ug)); };
    auto issue = [&](int kk, Staged& s) {
        s.kw = kk;
        if (kk < 0 || kk >= n2) s.kw = per_z ? ((kk % n2) + n2) % n2 : -1;
        if (s.kw >= 0) {
            const size_t off = (size_t)s.kw * plane;
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                if (act[r]) s.o[r] = ld.load_own(off + base0 + (size_t)r * n0);
                else if constexpr (Ld::PLAIN) s.o[r].a = bpair(i, jrow + r, s.kw);
            }
            if constexpr (requires { ld.prefetch_own((size_t)0); }) {
                // The demand loads run one plane ahead in registers (two planes spill); with one CTA per SM that is
                // ~50 KB in flight per SM, marginal against the HBM latency.  One lane per 128 bytes also pulls the
                // plane after that into L2 (no register): cg_pass_a 1.447 -> 1.321 ms at 512^3 (distance 2: 1.333,
                // 3: 1.380, 4: no gain).  The same two lines made the register-capped fused SOR kernel 20 % slower.
                if ((lx & 7) == 0 && s.kw + 1 < n2) {
#pragma unroll
                    for (int r = 0; r < RPT; ++r)
                        if (act[r]) ld.prefetch_own(off + plane + base0 + (size_t)r * n0);
                }
            }
#pragma unroll
            for (int m = 0; m < NH; ++m) {
                if (hcls[m] == 1) s.h[m] = ld.load(off + (size_t)hwj[m] * n0 + hwi[m]);
                else if constexpr (Ld::PLAIN) { if (hcls[m] == 2) s.h[m].a = bpair(hi[m], hj[m], s.kw); }
            }
        } else if constexpr (Ld::PLAIN) {
#pragma unroll
            for (int r = 0; r < RPT; ++r) s.o[r].a = bpair(i, jrow + r, kk);
        }
    };
    auto push = [&](int r, double2 v) {  // z register queue: zq[r][m] = plane (newest - 2R + m) of owned row r
        if constexpr (ZQ) {
#pragma unroll
            for (int m = 0; m < 2 * R; ++m) zq[r][m] = zq[r][m + 1];
            zq[r][2 * R] = v;
        }
    };
    auto commit = [&](int kk, const Staged& s) {
        double* slot = ring + ((kk + 2 * NS) & (NS - 1)) * SLOT;
        if constexpr (Ld::PLAIN) {
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                st2(slot + so0 + r * SW, s.o[r].a);
                push(r, s.o[r].a);
            }
            if (s.kw >= 0) {
#pragma unroll
                for (int m = 0; m < NH; ++m)
                    if (hcls[m] != 0) st2(slot + hso[m], s.h[m].a);
            }
        } else if (s.kw >= 0) {
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                double2 fv;
                if (act[r]) {
                    if constexpr (Ld::USES_DIAG) {
                        // the row diagonals of the two owned points from the coefficients already in registers
                        // (same expressions as stencil.cuh row_diag, so the quotients are the same bits)
                        double d0, d1;
                        if constexpr (sph_rd) {
                            fv = ld.form_own_rd(s.o[r], odv[r][0], odv[r][1], ord_[r][0], ord_[r][1]);
                            d0 = d1 = 0.0;
                        } else if constexpr (KIND == KIND_SPH) {
                            d0 = fma(rc.ir2[0], rc.dt[r], rc.dr[0]);
                            d1 = fma(rc.ir2[1], rc.dt[r], rc.dr[1]);
                        } else if constexpr (KIND == KIND_CART6) {
                            d0 = d1 = rc.d;
                        } else {
                            d0 = rc.plain ? rc.d : row_diag<double, KIND_CART2>(op, i, jrow + r, s.kw);
                            d1 = rc.plain ? rc.d : row_diag<double, KIND_CART2>(op, i + 1, jrow + r, s.kw);
                        }
                        if constexpr (!sph_rd) fv = ld.form_own(s.o[r], d0, d1);
                    } else {
                        fv = ld.form(op, s.o[r], i, jrow + r, s.kw);
                    }
                    if constexpr (Ld::SIDE) {
                        if (kk >= k0 && kk < k1) ld.side(s.o[r], (size_t)s.kw * plane + base0 + (size_t)r * n0);
                    }
                } else {
                    fv = bpair(i, jrow + r, s.kw);
                }
                st2(slot + so0 + r * SW, fv);
                push(r, fv);
            }
#pragma unroll
            for (int m = 0; m < NH; ++m) {
                if (hcls[m] == 1)
                {
                    if constexpr (Ld::USES_DIAG && KIND == KIND_SPH)
                    {
                        if constexpr (sph_rd)
                            st2(slot + hso[m], ld.form_own_rd(s.h[m], hd0[m], hd1[m], 1.0 / hd0[m], 1.0 / hd1[m]));
                        else
                            st2(slot + hso[m], ld.form_own(s.h[m], hd0[m], hd1[m]));  // spherical diagonal: no k dependence
                    }
                    else
                        st2(slot + hso[m], ld.form(op, s.h[m], hwi[m], hwj[m], s.kw));
                }
                else if (hcls[m] == 2)
                    st2(slot + hso[m], bpair(hi[m], hj[m], s.kw));
            }
        } else {
            // plane beyond a non-periodic z face: zeros (or a wrapped tiny grid); only owned columns are ever read
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                const double2 fv = bpair(i, jrow + r, kk);
                st2(slot + so0 + r * SW, fv);
                push(r, fv);
            }
        }
    };

    // prologue: planes k0-R .. k0+R-1, two at a time
    for (int kk = k0 - R; kk < k0 + R; kk += 2) {
        Staged a, b;
        issue(kk, a);
        issue(kk + 1, b);
        commit(kk, a);
        commit(kk + 1, b);
    }
    Staged st[PF];
    typename Ep::Raw est[PF][RPT];
#pragma unroll
    for (int u = 0; u < PF; ++u) {
        issue(k0 + R + u, st[u]);
        if (k0 + u < k1) {
#pragma unroll
            for (int r = 0; r < RPT; ++r)
                if (act[r]) est[u][r] = ep.load((size_t)(k0 + u) * plane + base0 + (size_t)r * n0);
        }
    }

    for (int kb = k0; kb < k1; kb += PF) {
#pragma unroll
        for (int u = 0; u < PF; ++u) {
            const int k = kb + u;
            if (k >= k1) break;  // uniform over the CTA
            commit(k + R, st[u]);
            typename Ep::Raw ecur[RPT];
#pragma unroll
            for (int r = 0; r < RPT; ++r) ecur[r] = est[u][r];
            if (k + PF < k1) {
                issue(k + PF + R, st[u]);
#pragma unroll
                for (int r = 0; r < RPT; ++r)
                    if (act[r]) est[u][r] = ep.load((size_t)(k + PF) * plane + base0 + (size_t)r * n0);
            }
            __syncthreads();
            const double* c0p = ring + ((k + 2 * NS) & (NS - 1)) * SLOT + so0;
            // radius 3: the y window of all owned rows (rows jrow-3 .. jrow+RPT+2), read once; owned rows from the z queue
            double2 yw[KIND == KIND_CART6 ? RPT + 6 : 1];
            if constexpr (KIND == KIND_CART6 && Cfg::YW != 0) {
#pragma unroll
                for (int m = 0; m < RPT + 6; ++m) {
                    if (ZQ && m >= 3 && m < RPT + 3)
                        yw[m] = zq[ZQ ? m - 3 : 0][R];
                    else
                        yw[m] = ld2(c0p + (m - 3) * SW);
                }
            }
#pragma unroll
            for (int r = 0; r < RPT; ++r) {
                if (!act[r]) continue;
                const double* P = c0p + r * SW;
                const int o = so0 + r * SW;
                double2 C;
                if constexpr (KIND == KIND_CART6 && Cfg::YW != 0)
                    C = yw[r + 3];
                else
                    C = ld2(P);
                double2 lv;
                if constexpr (KIND == KIND_CART6) {
                    const double2 xa = ld2(P - 4), xb = ld2(P - 2), xc = ld2(P + 2), xd = ld2(P + 4);
                    double2 t0, t1, t2;
                    {
                        // point i: -1 xb.y, +1 C.y, -2 xb.x, +2 xc.x, -3 xa.y, +3 xc.y ; point i+1 shifted by one
                        double w = 1.5 * (xb.y + C.y);
                        w = fma(-3.0 / 20.0, xb.x + xc.x, w);
                        t0.x = fma(1.0 / 90.0, xa.y + xc.y, w);
                        w = 1.5 * (C.x + xc.x);
                        w = fma(-3.0 / 20.0, xb.y + xc.y, w);
                        t0.y = fma(1.0 / 90.0, xb.x + xd.x, w);
                    }
                    {
                        // rows r-3 .. r+3 out of the window read once per plane for all owned rows
                        double2 m1, p1, m2, p2, m3, p3;
                        if constexpr (Cfg::YW != 0) {
                            m1 = yw[r + 2]; p1 = yw[r + 4]; m2 = yw[r + 1]; p2 = yw[r + 5]; m3 = yw[r]; p3 = yw[r + 6];
                        } else {
                            m1 = ld2(P - SW); p1 = ld2(P + SW); m2 = ld2(P - 2 * SW); p2 = ld2(P + 2 * SW);
                            m3 = ld2(P - 3 * SW); p3 = ld2(P + 3 * SW);
                        }
                        double w = 1.5 * (m1.x + p1.x);
                        w = fma(-3.0 / 20.0, m2.x + p2.x, w);
                        t1.x = fma(1.0 / 90.0, m3.x + p3.x, w);
                        w = 1.5 * (m1.y + p1.y);
                        w = fma(-3.0 / 20.0, m2.y + p2.y, w);
                        t1.y = fma(1.0 / 90.0, m3.y + p3.y, w);
                    }
                    {
                        double2 m1, p1, m2, p2, m3, p3;
                        if constexpr (ZQ) {
                            m1 = zq[r][2]; p1 = zq[r][4]; m2 = zq[r][1]; p2 = zq[r][5]; m3 = zq[r][0]; p3 = zq[r][6];
                        } else {
                            m1 = ld2(ring + ((k - 1 + 2 * NS) & (NS - 1)) * SLOT + o);
                            p1 = ld2(ring + ((k + 1 + 2 * NS) & (NS - 1)) * SLOT + o);
                            m2 = ld2(ring + ((k - 2 + 2 * NS) & (NS - 1)) * SLOT + o);
                            p2 = ld2(ring + ((k + 2 + 2 * NS) & (NS - 1)) * SLOT + o);
                            m3 = ld2(ring + ((k - 3 + 2 * NS) & (NS - 1)) * SLOT + o);
                            p3 = ld2(ring + ((k + 3 + 2 * NS) & (NS - 1)) * SLOT + o);
                        }
                        double w = 1.5 * (m1.x + p1.x);
                        w = fma(-3.0 / 20.0, m2.x + p2.x, w);
                        t2.x = fma(1.0 / 90.0, m3.x + p3.x, w);
                        w = 1.5 * (m1.y + p1.y);
                        w = fma(-3.0 / 20.0, m2.y + p2.y, w);
                        t2.y = fma(1.0 / 90.0, m3.y + p3.y, w);
                    }
                    double s = t0.x * rc.c0;
                    s = fma(t1.x, rc.c1, s);
                    s = fma(t2.x, rc.c2, s);
                    lv.x = fma(-rc.d, C.x, s);
                    s = t0.y * rc.c0;
                    s = fma(t1.y, rc.c1, s);
                    s = fma(t2.y, rc.c2, s);
                    lv.y = fma(-rc.d, C.y, s);
                } else {
                    const double2 xl = ld2(P - 2), xr = ld2(P + 2);
                    const double2 ym = ld2(P - SW), yp = ld2(P + SW);
                    const double2 zm = ld2(ring + ((k - 1 + 2 * NS) & (NS - 1)) * SLOT + o),
                                  zp = ld2(ring + ((k + 1 + 2 * NS) & (NS - 1)) * SLOT + o);
                    if constexpr (KIND == KIND_CART2) {
                        double d0 = rc.d, d1 = rc.d;
                        if (!rc.plain) {
                            d0 = row_diag<double, KIND_CART2>(op, i, jrow + r, k);
                            d1 = row_diag<double, KIND_CART2>(op, i + 1, jrow + r, k);
                        }
                        double s = (xl.y + C.y) * rc.c0;
                        s = fma(ym.x + yp.x, rc.c1, s);
                        s = fma(zm.x + zp.x, rc.c2, s);
                        lv.x = fma(-d0, C.x, s);
                        s = (C.x + xr.x) * rc.c0;
                        s = fma(ym.y + yp.y, rc.c1, s);
                        s = fma(zm.y + zp.y, rc.c2, s);
                        lv.y = fma(-d1, C.y, s);
                    } else {
                        // spherical row (stencil.cuh row_offsum / row_diag, KIND_SPH)
                        double s = rc.arm[0] * xl.y;
                        s = fma(rc.arp[0], C.y, s);
                        double t = rc.atm[r] * ym.x;
                        t = fma(rc.atp[r], yp.x, t);
                        t = fma(rc.cp[r], zm.x + zp.x, t);
                        double off = fma(rc.ir2[0], t, s);
                        lv.x = fma(-fma(rc.ir2[0], rc.dt[r], rc.dr[0]), C.x, off);
                        s = rc.arm[1] * C.x;
                        s = fma(rc.arp[1], xr.x, s);
                        t = rc.atm[r] * ym.y;
                        t = fma(rc.atp[r], yp.y, t);
                        t = fma(rc.cp[r], zm.y + zp.y, t);
                        off = fma(rc.ir2[1], t, s);
                        lv.y = fma(-fma(rc.ir2[1], rc.dt[r], rc.dr[1]), C.y, off);
                    }
                }
                ep.apply(ecur[r], (size_t)k * plane + base0 + (size_t)r * n0, i, jrow + r, k, C, lv, acc);
            }
        }
    }
    }  // segments
    if constexpr (Ep::NRED > 0) {
        double vals[Ep::NRED];
#pragma unroll
        for (int r = 0; r < Ep::NRED; ++r) vals[r] = acc[r];
        grid_reduce<Ep::NRED>(vals, rb, [&](const double* t) { ep.finish(t); });
    }
}

// How one launch is cut into runs of (tile, plane) items, and what it is expected to cost (arbitrary time unit:
// planes x rows of the tile, per wave).
struct PlanePlan {
    long items = 0, nctas = 0;
    int per_tile = 0, ntx = 0;
    double cost = 1e300;
};

// Two ways to schedule: whole z chunks (per_tile runs per tile, all tiles march z together, so the xy halo of a tile is
// still in L2 when its neighbour asks for it) or one linear split into equal runs (all SMs busy for any grid, but
// neighbouring tiles drift apart in z and their halos come from HBM again: measured +22 % DRAM traffic on the 512^3
// 19-point CG pass).  The linear split therefore carries a penalty and wins only when chunks leave SMs idle.
template <class G>
static PlanePlan plane_plan(const Op& op, long slots, int force_split /* POISSON_OPT_PLANE_SPLIT: 1 always, 0 never, -1 auto */) {
    PlanePlan pl;
    pl.ntx = (op.n[0] + G::TX - 1) / G::TX;
    const int nty = (op.n[1] + G::TY - 1) / G::TY;
    const long total = (long)pl.ntx * nty * op.n[2];
    const double halo_pen = force_split >= 0 ? (force_split ? 1e-3 : 1e3) : 1.0 + 0.15 * G::R;
    pl.items = std::max(4L, (total + slots - 1) / slots);
    pl.nctas = (total + pl.items - 1) / pl.items;
    pl.per_tile = 0;
    pl.cost = ((double)pl.items + 2.0 * (G::R + 1) + 4.0) * G::TY * halo_pen;
    for (int nz = 1; nz <= op.n[2]; ++nz) {
        const int kc = (op.n[2] + nz - 1) / nz;
        if (kc < 4 && nz > 1) break;
        const int nzz = (op.n[2] + kc - 1) / kc;
        const long ctas = (long)pl.ntx * nty * nzz;
        const double cost = (double)((ctas + slots - 1) / slots) * (kc + G::R + 1.0) * G::TY;
        if (cost < pl.cost - 1e-9) {
            pl.cost = cost;
            pl.items = kc;
            pl.per_tile = nzz;
            pl.nctas = ctas;
        }
    }
    return pl;
}

template <int KIND, class Cfg, class Ld, class Ep>
static int plane_resident(poisson_ctx* ctx, int* out) {
    using G = PlaneGeom<KIND, Cfg>;
    auto kern = k_plane<KIND, Cfg, Ld, Ep>;
    int resident = 0;
    const int rc = kernel_ready(ctx, kern, G::NT, G::SMEM, &resident);
    if (rc != POISSON_OK) return rc;
    if (resident < 1) return fail(ctx, POISSON_CUDA_ERROR, "plane kernel does not fit on an SM");
    *out = resident;
    return POISSON_OK;
}

template <int KIND, class Cfg, class Ld, class Ep>
static int plane_run(poisson_ctx* ctx, const Op& op, const Ld& ld, const Ep& ep, bool ug, int kid, const PlanePlan& pl) {
    using G = PlaneGeom<KIND, Cfg>;
    const dim3 g((unsigned)pl.nctas), b(G::NTX, G::NTY);
    if ((size_t)g.x > (size_t)kMaxRedBlocks) return fail(ctx, POISSON_UNSUPPORTED, "grid too large");
    pre_launch(ctx, kid);
    k_plane<KIND, Cfg, Ld, Ep><<<g, b, G::SMEM, ctx->stream>>>(op, ld, ep, pl.items, pl.per_tile, pl.ntx, ug, ctx->red);
    post_launch(ctx, kid);
    return POISSON_OK;
}

// Tile: 128 x 16 points, two rows per thread, one CTA per SM (measured on B200: 64 x 16 with two CTAs per SM, one or
// four rows per thread, a register queue for the z neighbours, 128 x 14 tiles — exactly 148 of them on a 512^2 plane —
// and two-plane prefetch were all slower).
using CfgA = TileCfg<128, 16, 2, 1, 1>;

template <int KIND, class Ld, class Ep>
static int launch_plane(poisson_ctx* ctx, const Op& op, const Ld& ld, const Ep& ep, bool ug, int kid) {
    int ra = 0, rc;
    if ((rc = plane_resident<KIND, CfgA, Ld, Ep>(ctx, &ra)) != POISSON_OK) return rc;
    const PlanePlan pa = plane_plan<PlaneGeom<KIND, CfgA>>(op, (long)ctx->num_sms * ra, ctx->opt_plane_split);
    return plane_run<KIND, CfgA, Ld, Ep>(ctx, op, ld, ep, ug, kid, pa);
}

// The plane engine needs 16-byte aligned pairs: even n0 (every row then starts on a pair boundary).
static inline bool plane_eligible(const poisson_ctx* ctx, const Op& op) {
    if (ctx->opt_path == 1) return false;
    if (op.n[0] % 2 != 0) return false;
    if (ctx->opt_path == 2) return true;
    return op.n[0] >= 64 && (size_t)op.n[0] * op.n[1] * op.n[2] >= (size_t)1 << 19;
}

}  // namespace pb
