// batch.cu — step a3 for P > 1 parameter points: the amplitude combine as the dense complex contraction it is,
//   A_xi(p, i) = sum_e C(p, e) B_{e,xi}(i),      S(p, i) = |A_+|^2 + |A_-|^2,
// on the FP64 tensor cores (mma.sync.m8n8k4.f64 — DMMA; tcgen05 has no f64 kind), fused with the -log L /
// normalisation reduction (a5).  Eqs. 4, 5, 10, 12.
//
// Realified GEMM, rows = parameter points, columns = events, contraction index = (basis entry, re/im):
//   Re A(p) = sum_e  c_re(p,e) b_re(e) - c_im(p,e) b_im(e)      (m-tile "RE" of a point octet)
//   Im A(p) = sum_e  c_im(p,e) b_re(e) + c_re(p,e) b_im(e)      (m-tile "IM" of the same octet)
// so the real and imaginary parts of one (point, event) pair land in the same thread and |A|^2 needs no shuffle.
// A warp owns 16 points (two octets = four m-tiles) and keeps their coefficient fragments in registers for the
// whole kernel; the basis tile B (events x entries, both muon helicities) is formed on the fly from the
// lineshape columns and the kinematics cache into shared memory and read as B fragments by all eight warps.
//
// Extended basis: a point that moves a resonance's mass or width uses another lineshape column for that
// resonance's slots.  Those (column, slot) pairs are appended as extra basis entries after the K base entries;
// the coefficient matrix is block-sparse there, and only the (k-tile, octet) blocks that are non-zero are
// multiplied (the per-warp item list), so a MINUIT-style gradient batch costs ~10 % more than the base GEMM.
#include "tile_basis.cuh"

namespace amp {

template <int NKT, int MODE>
__global__ void __launch_bounds__(BT_THREADS, 1) k_batch(const __grid_constant__ BatchArgs a) {
    extern __shared__ __align__(16) double smem[];
    const int KP = a.nent * 2;                                 // realified rows (multiple of 4)
    const TileSmem t = carve_tile_smem(smem, KP, a.ncolu);
    double* const Bs = t.Bs;
    double* const ws = t.ws;
    double* const sw = t.sw;
    double* const sang = t.sang;
    double2* const scol = t.scol;
    uint64_t* const full = t.full;
    const int nang = a.have_z ? BT_NANG : 6;
    const bool with_w = MODE == MODE_NORM;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // coefficient fragments of this warp's 16 points: [octet][re/im][k-tile]
    double Afr[2][2][NKT];
#pragma unroll
    for (int o = 0; o < 2; ++o)
#pragma unroll
        for (int ri = 0; ri < 2; ++ri)
#pragma unroll
            for (int kt = 0; kt < NKT; ++kt) Afr[o][ri][kt] = a.Adense[((((size_t)(2 * warp + o) * 2 + ri) * NKT) + kt) * 32 + lane];
    const int it0 = a.item_start[warp], it1 = a.item_start[warp + 1];
    const int prow = lane >> 2;                                // point row within an octet
    // row -> parameter point (the host spreads the points that own extended-basis blocks evenly over the warps)
    const int pt0 = a.point_of_row[16 * warp + prow], pt1 = a.point_of_row[16 * warp + 8 + prow];
    const bool live0 = pt0 >= 0, live1 = pt1 >= 0;
    const bool warp_live = __any_sync(0xffffffffu, live0 || live1);

    double sum[2] = {0.0, 0.0}, prod[2] = {1.0, 1.0};
    bool bad = false;
    const long long ntiles = (a.n + BT_EVENTS - 1) / BT_EVENTS;
    if (tid == 0) {
        bmbar_init(full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    stage_tile_entries(a, t);
    __syncthreads();
    if (tid == 0 && (long long)blockIdx.x < ntiles) issue_stage(a, blockIdx.x, scol, sang, sw, full, nang, with_w);
    uint32_t parity = 0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x, parity ^= 1) {
        // ---- basis tile from the staged inputs: thread (part, ev) fills entries part, part+4, ... of event ev, both helicities
        bmbar_wait(full, parity);
        build_basis_tile(a, t, tile, KP, with_w);
        __syncthreads();   // basis tile complete, staging area consumed: stream the next tile into it during the DMMA phase
        if (tid == 0 && tile + gridDim.x < ntiles) issue_stage(a, tile + gridDim.x, scol, sang, sw, full, nang, with_w);
        // ---- DMMA: this warp's 16 points x 64 events x both helicities
#pragma unroll 1
        for (int nt = 0; nt < (warp_live ? BT_EVENTS / 8 : 0); ++nt) {
            // both helicities side by side: eight independent accumulator chains per warp keep the DMMA pipe fed
            double acc[2][2][2][2];   // [xi][octet][re/im][event pair]
#pragma unroll
            for (int xi = 0; xi < 2; ++xi)
#pragma unroll
                for (int o = 0; o < 2; ++o)
#pragma unroll
                    for (int ri = 0; ri < 2; ++ri) acc[xi][o][ri][0] = acc[xi][o][ri][1] = 0.0;
            const double* bbase = Bs + (size_t)(lane & 3) * BT_STRIDE + 8 * nt + (lane >> 2);
            const size_t xoff = (size_t)KP * BT_STRIDE;
#pragma unroll
            for (int kt = 0; kt < NKT; ++kt) {
                const double bP = bbase[(size_t)4 * kt * BT_STRIDE], bM = bbase[xoff + (size_t)4 * kt * BT_STRIDE];
                dmma884(acc[0][0][0], Afr[0][0][kt], bP);
                dmma884(acc[1][0][0], Afr[0][0][kt], bM);
                dmma884(acc[0][0][1], Afr[0][1][kt], bP);
                dmma884(acc[1][0][1], Afr[0][1][kt], bM);
                dmma884(acc[0][1][0], Afr[1][0][kt], bP);
                dmma884(acc[1][1][0], Afr[1][0][kt], bM);
                dmma884(acc[0][1][1], Afr[1][1][kt], bP);
                dmma884(acc[1][1][1], Afr[1][1][kt], bM);
            }
            for (int it = it0; it < it1; ++it) {           // non-zero blocks of the extended (variant) basis
                const int2 item = a.items[it];               // (first realified row of the k-tile, octet 0/1 of this warp)
                const double bP = bbase[(size_t)item.x * BT_STRIDE], bM = bbase[xoff + (size_t)item.x * BT_STRIDE];
                const double are = a.itemA[((size_t)it * 2) * 32 + lane], aim = a.itemA[((size_t)it * 2 + 1) * 32 + lane];
                if (item.y == 0) {
                    dmma884(acc[0][0][0], are, bP); dmma884(acc[1][0][0], are, bM);
                    dmma884(acc[0][0][1], aim, bP); dmma884(acc[1][0][1], aim, bM);
                } else {
                    dmma884(acc[0][1][0], are, bP); dmma884(acc[1][1][0], are, bM);
                    dmma884(acc[0][1][1], aim, bP); dmma884(acc[1][1][1], aim, bM);
                }
            }
            double S[2][2];
#pragma unroll
            for (int o = 0; o < 2; ++o)
#pragma unroll
                for (int j = 0; j < 2; ++j)
                    S[o][j] = fma(acc[0][o][0][j], acc[0][o][0][j], fma(acc[0][o][1][j], acc[0][o][1][j],
                              fma(acc[1][o][0][j], acc[1][o][0][j], acc[1][o][1][j] * acc[1][o][1][j])));
            const double w0 = ws[8 * nt + 2 * (lane & 3)], w1 = ws[8 * nt + 2 * (lane & 3) + 1];
            if (MODE == MODE_NORM) {
#pragma unroll
                for (int o = 0; o < 2; ++o) {
                    bad |= !isfinite(S[o][0]) || !isfinite(S[o][1]);
                    sum[o] = fma(w0, S[o][0], fma(w1, S[o][1], sum[o]));
                }
            } else {
                // sum of logs: multiply four S values (two events x two n-tiles), one log per product
#pragma unroll
                for (int o = 0; o < 2; ++o) {
                    const bool live = o ? live1 : live0;
                    const double s0 = (live && w0 > 0.0) ? S[o][0] : 1.0, s1 = (live && w1 > 0.0) ? S[o][1] : 1.0;
                    bad |= !(s0 > 0.0) || !(s1 > 0.0) || !isfinite(s0) || !isfinite(s1);
                    prod[o] *= s0 * s1;
                    if (nt & 1) { sum[o] += log(prod[o]); prod[o] = 1.0; }
                }
            }
        }
        __syncthreads();
    }
    if (bad) atomicOr(a.flag, 2);
    // the four lanes of a row hold different events of the same point: fixed xor tree, then one partial per (point, CTA)
#pragma unroll
    for (int o = 0; o < 2; ++o) {
        double v = sum[o];
        v += __shfl_xor_sync(0xffffffffu, v, 1);
        v += __shfl_xor_sync(0xffffffffu, v, 2);
        const int p = o ? pt1 : pt0;
        if ((lane & 3) == 0 && p >= 0) a.partial[(size_t)p * a.partial_stride + blockIdx.x] = v;
    }
}

size_t batch_smem(int nent, int ncolu) { return tile_smem_bytes(nent, ncolu); }
bool batch_fits(int nent, int ncolu) { return ncolu <= BATCH_MAX_COLS && batch_smem(nent, ncolu) <= (size_t)224 * 1024; }

int batch_grid(long long n) {
    const long long ntiles = (n + BT_EVENTS - 1) / BT_EVENTS;
    return (int)(ntiles < 1 ? 1 : (ntiles > sm_count() ? sm_count() : ntiles));   // persistent: one CTA per SM
}

cudaError_t launch_batch(const BatchArgs& a, int grid, cudaStream_t s) {
    const size_t smem = batch_smem(a.nent, a.ncolu);
    cudaError_t e = cudaSuccess;
#define AMP_LAUNCH(NKT, M)                                                                                           \
    {                                                                                                                \
        static DeviceOnce attr_done;                                                                               \
        if (attr_done.first()) { e = cudaFuncSetAttribute(k_batch<NKT, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, 224 * 1024); } \
        if (e == cudaSuccess) k_batch<NKT, M><<<grid, BT_THREADS, smem, s>>>(a);                                     \
    }
    if (a.nkt != BATCH_NKT) return cudaErrorInvalidValue;
    if (a.mode == MODE_NORM) AMP_LAUNCH(BATCH_NKT, MODE_NORM) else AMP_LAUNCH(BATCH_NKT, MODE_DATA)
#undef AMP_LAUNCH
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace amp
