// k_apply_bulk.cu — 7-point Cartesian apply / residual (fp64, non-periodic) with the xy planes staged in shared memory
// by the Tensor Memory Accelerator (cp.async.bulk.tensor, SASS UTMALDG) instead of by the threads:
//   out = L v   or   out = rhs - L v   (+ fp32 copy, + sum(out^2), sum(out)).            PAPER.md:43-45 (Eq. 1), 55, 57.
// A CTA of 64 x 4 threads owns a 128 x 8 tile and marches z; four such CTAs share an SM.  One thread issues, per plane,
// ONE tensor copy of the (128+4) x (8+2) x 1 box (tile + halo; out-of-range parts are zero-filled by the hardware) into
// a ring of NS planes and arms the plane's mbarrier with the byte count; copies run PF planes ahead of their use, so
// ~4 x PF x 10 KB per SM are in flight without a staging register or an LSU load instruction.  Every thread owns a
// 16-byte pair in two adjacent rows, keeps planes k-1, k, k+1 of them in registers (read once from the ring when a plane
// lands; the residual variants read the right-hand side from the tile that rides in the same slot) and takes the x / y neighbours of plane k from the ring; threads on a Dirichlet face take that neighbour from
// the ghost-face array instead.  One __syncthreads per plane frees the oldest slot.  Arithmetic order = stencil.cuh
// row_apply<KIND_CART2>, results bit-identical to the other apply kernels.
// (A first version issued one 1 KB cp.async.bulk per tile row: 18 copies per plane cost ~3.6 k cycles of copy-engine
// time per plane and ran at 140 Gpoint/s; the single tensor copy removes that.)
#include <algorithm>
#include <cstdint>
#include <cstdlib>

#include "pairq.cuh"
#include "tma.cuh"

namespace pb {

namespace bulk {
// Tile configuration: TX x TY points per CTA (64 x TY/2 ... threads: TX/2 pairs x TY/2 row pairs), NS ring slots, copies
// PF planes ahead, MINB resident CTAs per SM asked of the compiler.
template <int TX_, int TY_, int NS_, int PF_, int MINB_>
struct Cfg {
    static constexpr int TX = TX_, TY = TY_, NS = NS_, PF = PF_, MINB = MINB_;
    static constexpr int SW = TX + 4, SH = TY + 2, NTX = TX / 2, NT = NTX * (TY / 2);
    static constexpr int BOX_BYTES = SW * SH * 8;
    static constexpr int SLOT = ((BOX_BYTES + 127) / 128) * 16;  // slot pitch in doubles, 128-byte aligned
    static constexpr int RHS_BYTES = TX * TY * 8;  // residual variants: the tile of the right-hand side, no halo
    // ring pitch in doubles: the box of v, then (residual variants) the right-hand side of the plane before it
    __host__ __device__ static constexpr int pitch(bool with_rhs) { return SLOT + (with_rhs ? TX * TY : 0); }
    __host__ __device__ static constexpr size_t smem(bool with_rhs) {
        return (size_t)NS * pitch(with_rhs) * sizeof(double) + NS * sizeof(uint64_t) + 128;
    }
};

}  // namespace bulk

struct BulkGeom {
    int ntx, nty;
    long items;
};

template <class C, int MODE, bool RED, bool PLAIN>
__global__ void __launch_bounds__(C::NT, C::MINB)
    k_apply7_bulk(const Op op, const __grid_constant__ CUtensorMap vmap, const __grid_constant__ CUtensorMap fmap,
                  double* __restrict__ out, float* __restrict__ out32, const bool ug_in, const BulkGeom g, RedBuf rb,
                  double* scal) {
    using namespace tma;
    constexpr int TX = C::TX, TY = C::TY, SW = C::SW, NS = C::NS, PF = C::PF, BOX_BYTES = C::BOX_BYTES;
    constexpr int SLOT = C::pitch(MODE != 0), FOFF = C::SLOT;  // the right-hand side tile sits FOFF doubles into a slot
    constexpr uint32_t TX_BYTES = BOX_BYTES + (MODE != 0 ? C::RHS_BYTES : 0);
    extern __shared__ unsigned char smraw0[];
    unsigned char* const smraw = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smraw0) + 127) & ~uintptr_t(127));
    double* const ring = reinterpret_cast<double*>(smraw);
    uint64_t* const full = reinterpret_cast<uint64_t*>(ring + (size_t)NS * SLOT);
    const int n0 = op.n[0], n1 = op.n[1], n2 = op.n[2];
    const int tid = threadIdx.x, lx = tid % C::NTX, ty = tid / C::NTX;
    const bool ug = ug_in && op.gamma == 0.0;
    const double c0 = op.c[0], c1 = op.c[1], c2 = op.c[2];
    const double dplain = 2.0 * ((c0 + c1) + c2);
    const size_t plane = (size_t)n0 * n1;
    // ghost-face arrays of the Dirichlet faces in use (nullptr: that neighbour is zero, which is what the copy delivers)
    const double* gf[6];
#pragma unroll
    for (int f = 0; f < 6; ++f) gf[f] = (ug && op.bc[f] == POISSON_BC_DIRICHLET_GHOST) ? op.ghost[f] : nullptr;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    unsigned issued = 0, used = 0;  // planes issued / consumed so far: slot = count % NS, parity = (count / NS) & 1
    double s2 = 0.0, s1 = 0.0;

    const long total = (long)g.ntx * g.nty * n2;
    long pos = (long)blockIdx.x * g.items;
    const long end = min(total, pos + g.items);
    while (pos < end) {
        const int t = (int)(pos / n2), k0 = (int)(pos % n2);
        const int k1 = (int)min((long)n2, (long)k0 + (end - pos));
        pos += k1 - k0;
        const int i0 = (t % g.ntx) * TX, j0 = (t / g.ntx) * TY;
        const int i = i0 + 2 * lx, jr = j0 + 2 * ty;  // this thread's pair (i, i+1) in rows jr, jr+1
        const bool own0 = i < n0 && jr < n1, own1 = i < n0 && jr + 1 < n1;
        const int kbeg = k0 - 1, kend = k1;
        auto issue = [&](int kk) {  // thread 0: one tensor copy = tile + halo of plane kk (zero fill outside the array)
            if (tid == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                mbar_arrive_expect_tx(&full[issued % NS], TX_BYTES);
                tma_box(ring + (size_t)(issued % NS) * SLOT, &vmap, i0 - 2, j0 - 1, kk, &full[issued % NS]);
                // the plane that is computed when v(kk) lands is kk - 1: its right-hand side rides in the same slot
                if (MODE != 0) tma_box(ring + (size_t)(issued % NS) * SLOT + FOFF, &fmap, i0, j0, kk - 1, &full[issued % NS]);
            }
            ++issued;
        };
        double dx0 = dplain, dy0 = dplain, dx1 = dplain, dy1 = dplain;
        if (!PLAIN) {
            if (own0) { dx0 = a7_diag_xy<double>(op, i, jr); dy0 = a7_diag_xy<double>(op, i + 1, jr); }
            if (own1) { dx1 = a7_diag_xy<double>(op, i, jr + 1); dy1 = a7_diag_xy<double>(op, i + 1, jr + 1); }
        }
        for (int m = 0; m < PF && kbeg + m <= kend; ++m) issue(kbeg + m);
        const size_t cb0 = (size_t)jr * n0 + i, cb1 = cb0 + n0;
        double2 qm0 = make_double2(0, 0), qc0 = qm0, qp0 = qm0, qm1 = qm0, qc1 = qm0, qp1 = qm0;
        const int fo = FOFF + (2 * ty) * TX + 2 * lx;   // own pair of row jr in the right-hand side tile; row jr+1 is TX further
        const int so = (1 + 2 * ty) * SW + 2 + 2 * lx;  // own pair of row jr inside a slot; row jr+1 is SW further
        const double* prev = ring;                       // slot of the previous plane
        for (int kin = kbeg; kin <= kend; ++kin) {
            const double* const cur = ring + (size_t)(used % NS) * SLOT;
            mbar_wait(&full[used % NS], (used / NS) & 1u);
            ++used;
            qm0 = qc0; qc0 = qp0; qm1 = qc1; qc1 = qp1;
            qp0 = *reinterpret_cast<const double2*>(cur + so);
            qp1 = *reinterpret_cast<const double2*>(cur + so + SW);
            if (kin < 0 || kin >= n2) {  // a z ghost plane: the copy delivered zeros; owned pairs come from the face array
                const double* zf = kin < 0 ? gf[4] : gf[5];
                if (zf && own0) qp0 = *reinterpret_cast<const double2*>(zf + cb0);
                if (zf && own1) qp1 = *reinterpret_cast<const double2*>(zf + cb1);
            }
            const int k = kin - 1;
            if (k >= k0 && k < k1) {
                const double* const P = prev + so;
                double2 ya = *reinterpret_cast<const double2*>(P - SW), yb = *reinterpret_cast<const double2*>(P + 2 * SW);
                double xl0 = P[-1], xr0 = P[2], xl1 = P[SW - 1], xr1 = P[SW + 2];
                double2 below0 = qc1;  // neighbour of row jr in +y: own row jr+1 unless that is the ghost row
                if (i == 0 && gf[0]) { xl0 = gf[0][(size_t)k * n1 + jr]; if (own1) xl1 = gf[0][(size_t)k * n1 + jr + 1]; }
                if (i + 2 == n0 && gf[1]) { xr0 = gf[1][(size_t)k * n1 + jr]; if (own1) xr1 = gf[1][(size_t)k * n1 + jr + 1]; }
                if (jr == 0 && gf[2] && own0) ya = *reinterpret_cast<const double2*>(gf[2] + (size_t)k * n0 + i);
                if (jr + 2 == n1 && gf[3] && own0) yb = *reinterpret_cast<const double2*>(gf[3] + (size_t)k * n0 + i);
                if (jr + 1 == n1 && gf[3] && own0) below0 = *reinterpret_cast<const double2*>(gf[3] + (size_t)k * n0 + i);
                double2 fa = make_double2(0, 0), fb = fa;
                if (MODE != 0) {
                    fa = *reinterpret_cast<const double2*>(cur + fo);
                    fb = *reinterpret_cast<const double2*>(cur + fo + TX);
                }
                double dz00 = dx0, dz01 = dy0, dz10 = dx1, dz11 = dy1;
                if (!PLAIN && (k == 0 || k == n2 - 1)) {
                    dz00 = a7_diag_z<double>(op, dz00, k); dz01 = a7_diag_z<double>(op, dz01, k);
                    dz10 = a7_diag_z<double>(op, dz10, k); dz11 = a7_diag_z<double>(op, dz11, k);
                }
                const size_t po = (size_t)k * plane;
                auto finish = [&](double lv0, double lv1, double2 f, size_t q) {
                    const double o0 = MODE ? f.x - lv0 : lv0, o1 = MODE ? f.y - lv1 : lv1;
                    if (out) *reinterpret_cast<double2*>(out + q) = make_double2(o0, o1);
                    if (out32) *reinterpret_cast<float2*>(out32 + q) = make_float2((float)o0, (float)o1);
                    if (RED) {
                        s2 = fma(o0, o0, s2); s1 += o0;
                        s2 = fma(o1, o1, s2); s1 += o1;
                    }
                };
                if (own0) {  // row jr: y neighbours = ring row above (or ghost), row jr+1 (own, or ghost)
                    double s = (xl0 + qc0.y) * c0;
                    s = fma(ya.x + below0.x, c1, s);
                    s = fma(qm0.x + qp0.x, c2, s);
                    const double lv0 = fma(-dz00, qc0.x, s);
                    s = (qc0.x + xr0) * c0;
                    s = fma(ya.y + below0.y, c1, s);
                    s = fma(qm0.y + qp0.y, c2, s);
                    finish(lv0, fma(-dz01, qc0.y, s), fa, po + cb0);
                }
                if (own1) {  // row jr+1: y neighbours = own row jr, ring row below (or ghost)
                    double s = (xl1 + qc1.y) * c0;
                    s = fma(qc0.x + yb.x, c1, s);
                    s = fma(qm1.x + qp1.x, c2, s);
                    const double lv0 = fma(-dz10, qc1.x, s);
                    s = (qc1.x + xr1) * c0;
                    s = fma(qc0.y + yb.y, c1, s);
                    s = fma(qm1.y + qp1.y, c2, s);
                    finish(lv0, fma(-dz11, qc1.y, s), fb, po + cb1);
                }
            }
            prev = cur;
            __syncthreads();  // every reader is done with the planes before `cur`: their slots may be refilled
            if (kin + PF <= kend) issue(kin + PF);
        }
    }
    if (RED) {
        double vals[2] = {s2, s1};
        grid_reduce<2>(vals, rb, [=](const double* t) {
            scal[0] = t[0];
            scal[1] = t[1];
        });
    }
}

// ---- host side ----------------------------------------------------------------------------------------------------------
bool apply_bulk_ok(const poisson_ctx* ctx, const Op& op) {
    const int mode = ctx->opt_apply_bulk;  // POISSON_OPT_APPLY_BULK: 0 = never, 1 = whenever eligible; -1: large grids
    if (mode == 0 || ctx->opt_path == 1) return false;
    if (op.coord != POISSON_CARTESIAN || op.order != 2 || op.n[0] % 2 != 0) return false;
    for (int f = 0; f < 6; ++f)
        if (op.bc[f] == POISSON_BC_PERIODIC) return false;
    if (mode == 1) return true;
    return op.n[0] >= 128 && (size_t)op.n[0] * op.n[1] * op.n[2] >= (size_t)1 << 21;
}

template <class C, int MODE, bool RED>
static int bulk_launch(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, double* out, float* out32,
                       bool ug) {
    bool plain = op.gamma == 0.0;
    for (int f = 0; f < 6; ++f) plain = plain && op.bc[f] != POISSON_BC_NEUMANN0;
    BulkGeom g;
    g.ntx = (op.n[0] + C::TX - 1) / C::TX;
    g.nty = (op.n[1] + C::TY - 1) / C::TY;
    const long total = (long)g.ntx * g.nty * op.n[2];
    int resident = 0;
    CUtensorMap map, fmap;
    if (!tma::make_map3(v, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 8, op.n, C::SW, C::SH, &map)) return POISSON_UNSUPPORTED;  // the caller falls back to k_apply7
    fmap = map;
    if (MODE != 0 && !tma::make_map3(rhs, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 8, op.n, C::TX, C::TY, &fmap)) return POISSON_UNSUPPORTED;
    constexpr size_t SMEM = C::smem(MODE != 0);
    int rc = kernel_ready(ctx, k_apply7_bulk<C, MODE, RED, false>, C::NT, SMEM);
    if (rc == POISSON_OK) rc = kernel_ready(ctx, k_apply7_bulk<C, MODE, RED, true>, C::NT, SMEM, &resident);
    if (rc != POISSON_OK) return rc;
    if (resident < 1) resident = 1;
    g.items = std::max(4L, (total + (long)ctx->num_sms * resident - 1) / ((long)ctx->num_sms * resident));
    const int grid = (int)((total + g.items - 1) / g.items);
    if (grid > kMaxRedBlocks) return fail(ctx, POISSON_UNSUPPORTED, "grid too large for the reduction buffer");
    if (plain)
        PB_LAUNCH(ctx, KID_APPLY, (k_apply7_bulk<C, MODE, RED, true><<<grid, C::NT, SMEM, ctx->stream>>>(op, map, fmap, out, out32, ug, g, ctx->red, ctx->d_scal)));
    else
        PB_LAUNCH(ctx, KID_APPLY, (k_apply7_bulk<C, MODE, RED, false><<<grid, C::NT, SMEM, ctx->stream>>>(op, map, fmap, out, out32, ug, g, ctx->red, ctx->d_scal)));
    PB_CUDA_OK(cudaGetLastError());
    return POISSON_OK;
}

// Tile choice, measured at 256^3 on B200 (us per apply, MODE 0): 128 x 8 tiles with 4 CTAs per SM 58; 3 CTAs 63;
// 64 x 16 / 3 CTAs 66; 64 x 8 / 8 CTAs 64; 128 x 16 / 1 CTA of 512 threads 81 (= the thread-staged kernels): what pays
// is MANY SMALL CTAs per SM, so that one CTA's per-plane barrier is hidden behind the others.  The residual variants
// stage the right-hand side tile of the plane being computed in the same slot, by a second tensor copy on the same
// mbarrier (residual norm 68 us; with the threads loading it into a register queue one plane ahead it was 96 us: the
// queue rotation waits for the load, which leaves one plane per DRAM latency per CTA).  Ring of 4 / 3 CTAs per SM and
// ring of 3 / 4 CTAs measure the same; ring of 6 / 2 CTAs 82 us.
template <int MODE, bool RED>
static int bulk_cfg(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, double* out, float* out32,
                    bool ug) {
    using C4 = bulk::Cfg<128, 8, 5, 3, 4>;  // 256 threads, ring of 5 planes, copies 3 planes ahead, four CTAs per SM
    using C3 = bulk::Cfg<128, 8, 4, 3, 3>;  // 256 threads, ring of 4 planes (+ rhs tiles), copies 3 planes ahead, three CTAs per SM
    if (MODE == 0) return bulk_launch<C4, MODE, RED>(ctx, op, v, rhs, out, out32, ug);
    return bulk_launch<C3, MODE, RED>(ctx, op, v, rhs, out, out32, ug);
}

int apply_bulk(poisson_ctx* ctx, const Op& op, const double* v, const double* rhs, double* out, float* out32, int mode,
               bool ug, bool reduce) {
    if (mode == 0) return bulk_cfg<0, false>(ctx, op, v, rhs, out, out32, ug);
    if (!reduce) return bulk_cfg<1, false>(ctx, op, v, rhs, out, out32, ug);
    return bulk_cfg<1, true>(ctx, op, v, rhs, out, out32, ug);
}

}  // namespace pb
