// Dhop, warp-specialised TMA kernel for 4x4x4x4 tiles (the fast path on sm_100a).
//
// Persistent CTAs take tiles from a global in-order queue over an L2-friendly sweep order.  Per CTA:
//   * warp group 0 is the PRODUCER (one warp active, registers shrunk with setmaxnreg): for every
//     (tile, s) it fills one stage of an NST-deep shared-memory ring with the s-slice working set of
//     the tile -- 12 regions of [K][32 slots] 16-byte vectors:
//        regions 0-3   the tile's own four t-slabs           (TMA, 512-byte rows)
//        regions 4,5   +t / -t faces of the neighbour tiles  (TMA, 512-byte rows)
//        regions 6,7   +z / -z faces                         (TMA, 128-byte rows)
//        regions 8,9   +y / -y faces                         (fp32: TMA, 32-byte rows; fp64: cp.async gather)
//        regions 10,11 +x / -x faces                         (cp.async gather: the checkerboard makes the x
//                                                             face a row-parity pattern no box can describe)
//     all completing on the stage's `full` mbarrier; the next tile's links are prefetched into L2 with one bulk
//     prefetch issued with the tile's last slice;
//   * the other warp groups are CONSUMERS: each thread keeps its links in registers for the whole s
//     loop (third row rebuilt once per tile, antiperiodic sign folded in), waits on `full`, reads its
//     neighbours with 128-bit LDS at a uniform 512-byte k pitch, spin-projects, multiplies,
//     reconstruct-accumulates, releases the stage on the `empty` mbarrier and stores 128-bit
//     coalesced with a streaming hint.  No block-wide barrier inside the loop: warps drift apart and
//     keep the FP and shared-memory pipes busy at the same time.
// fp32: one thread per site (8 links in registers), 2 CTAs/SM.  fp64: two lanes (l, l^16) per site (forward legs
// on one, backward legs on the other), partial sums exchanged by warp shuffles, 1 CTA/SM; its fields use the
// XOR-rotated lane order of dwf_layout.cuh and conflict-free face slots (build_tma_tables_swz).
// EPI = 1 adds the last step of Mpc as an epilogue: out_s = Mee xin_s + scale (Dhop in)_s and its |.|^2.
// Register budget (232 per consumer thread) decides the rest: the fp32 plain kernel pins the rebuilt third link rows so that
// the compiler does not recompute them in every slice; the fp64 kernel with the epilogue does the opposite on purpose (rows
// 0, 1 resident, row 2 rebuilt per slice) to have registers for its epilogue loads.  Batched fields (N systems, fifth
// dimension N * Ls, dwf_internal.h) run through the same kernels with g.Ls = N * Ls; only the epilogue knows the physical Ls.
#include <cuda.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#include "dwf_dhop_math.cuh"

namespace dwf {

// ------------------------------------------------------------------------------------------ host tables
namespace {

constexpr int TSV = 128;      // sites of one parity in a 4^4 tile
constexpr int NREG = 12;      // regions per stage

struct TmaTables {
    std::vector<uint16_t> off;     // [2][8][128]  stage offset (16-byte units, k = 0) of the leg's neighbour
    std::vector<uint8_t> gsrc;     // [2][4][32]   gathered faces (+x, -x, +y, -y): source lane in the neighbour tile
    std::vector<uint16_t> gdst;    // [2][4][32]   ... and its stage offset (16-byte units, k = 0)
    std::vector<uint8_t> xsrc;     // [2][2][32]   plain order (fp32): source lane (in the +x / -x tile) of each x-face site
    std::vector<uint16_t> xdst;    // [2][2][32]   ... and its stage offset (16-byte units, k = 0)
};

inline int lane_of_plain(int tx, int ty, int tz, int tt) { return ((tt * 4 + tz) * 4 + ty) * 2 + (tx >> 1); }

// fp32 fields: plain lane order, +-y faces by TMA boxes, +-x faces gathered (the kernel has no registers for more).
// The gathered x faces are interleaved over regions 10 and 11 like in the fp64 scheme below (+x sites on the even bank
// groups 2 ty, -x sites on the odd ones 2 ty + 1: the groups the quarter warp's interior lanes leave free), which removes
// the x-leg bank conflicts; the y legs keep theirs (their faces are TMA boxes with a fixed layout).
TmaTables build_tma_tables_plain(int K) {
    TmaTables t;
    t.off.assign(2 * 8 * TSV, 0);
    t.xsrc.assign(2 * 2 * 32, 0);
    t.xdst.assign(2 * 2 * 32, 0);
    for (int p = 0; p < 2; ++p) {
        const int q = 1 - p;   // input parity
        int xslot[2][4][4][4];     // [f][tt][tz][ty] stage offset of the x-face site, f = 0: +x tile (tx = 0), 1: -x tile (tx = 3)
        int cnt[2][8], nface[2] = {0, 0};
        memset(cnt, 0, sizeof(cnt));
        for (int f = 0; f < 2; ++f)
            for (int tt = 0; tt < 4; ++tt)
                for (int tz = 0; tz < 4; ++tz)
                    for (int ty = 0; ty < 4; ++ty) {
                        xslot[f][tt][tz][ty] = -1;
                        const int tx = f ? 3 : 0;
                        if (((q + tx + ty + tz + tt) & 1) != 0) continue;
                        const int b = 2 * ty + f;
                        const int s64 = b + 8 * cnt[f][b]++;
                        const int o = (10 + (s64 >> 5)) * K * 32 + (s64 & 31);
                        xslot[f][tt][tz][ty] = o;
                        const int i = nface[f]++;
                        t.xsrc[(p * 2 + f) * 32 + i] = (uint8_t)lane_of_plain(tx, ty, tz, tt);
                        t.xdst[(p * 2 + f) * 32 + i] = (uint16_t)o;
                    }
        for (int tt = 0; tt < 4; ++tt)
            for (int tz = 0; tz < 4; ++tz)
                for (int ty = 0; ty < 4; ++ty)
                    for (int txh = 0; txh < 2; ++txh) {
                        const int tx = 2 * txh + ((p + ty + tz + tt) & 1);
                        const int lane = lane_of_plain(tx, ty, tz, tt);
                        for (int leg = 0; leg < 8; ++leg) {
                            const int mu = leg >> 1;
                            int y[4] = {tx, ty, tz, tt};
                            y[mu] += (leg & 1) ? -1 : +1;
                            int o;
                            if (y[mu] >= 0 && y[mu] < 4) {
                                o = y[3] * K * 32 + (y[2] * 4 + y[1]) * 2 + (y[0] >> 1);
                            } else {
                                const int up = (y[mu] >= 4);
                                y[mu] = (y[mu] + 4) & 3;
                                const int yh = y[0] >> 1;
                                if (mu == 3)      o = (up ? 4 : 5) * K * 32 + (y[2] * 4 + y[1]) * 2 + yh;
                                else if (mu == 2) o = (up ? 6 : 7) * K * 32 + y[3] * 8 + y[1] * 2 + yh;
                                else if (mu == 1) o = (up ? 8 : 9) * K * 32 + (y[3] * 4 + y[2]) * 2 + yh;
                                else              o = xslot[up ? 0 : 1][y[3]][y[2]][y[1]];
                            }
                            t.off[(p * 8 + leg) * TSV + lane] = (uint16_t)o;
                        }
                    }
    }
    return t;
}

// lane order of dwf_layout.cuh for 4^4 tiles: y rows XOR-rotated by tz
inline int lane_of(int tx, int ty, int tz, int tt) { return ((tt * 4 + tz) * 4 + (ty ^ tz)) * 2 + (tx >> 1); }

// Shared-memory slots.  A region is [K][32 slots] of 16-byte vectors, so slot mod 8 is the bank group of a 128-bit
// access.  With the XOR-rotated lane order the 8 lanes of a quarter warp (one (tz, tt), all ty, both tx halves) read,
// for every leg, 6 or 8 interior / TMA-written slots in distinct bank groups, and the face lanes miss exactly the
// groups 2 (ty ^ tz) + {0, 1} (y legs) or 2 (ty ^ tz) + (0: +x, 1: -x) (x legs).  The x and y faces are written by
// cp.async gathers, free to put every face site into a slot of exactly that group: the +-y faces in their own regions
// (4 sites per group), the +-x faces interleaved over regions 10 and 11 (+x the even groups, -x the odd ones, 8 sites
// per group).  Result: no shared-memory bank conflict on any leg (it was 1.44 wavefronts per ideal one).
// fp64 fields: XOR-rotated lane order, conflict-free slots (see above)
TmaTables build_tma_tables_swz(int K) {
    TmaTables t;
    t.off.assign(2 * 8 * TSV, 0);
    t.gsrc.assign(2 * 4 * 32, 0);
    t.gdst.assign(2 * 4 * 32, 0);
    for (int p = 0; p < 2; ++p) {
        const int q = 1 - p;   // input parity
        // ---- slots of the gathered faces: face f = 0 (+x: sites tx = 0 of the +x tile), 1 (-x: tx = 3), 2 (+y: ty = 0), 3 (-y: ty = 3)
        int slot_of[4][4][4][4];          // [f][tt][tz][u]: u = ty for x faces, tx/2 for y faces; -1 = not a site of parity q
        int cnt[4][8];
        memset(cnt, 0, sizeof(cnt));
        int nface[4] = {0, 0, 0, 0};
        for (int f = 0; f < 4; ++f)
            for (int tt = 0; tt < 4; ++tt)
                for (int tz = 0; tz < 4; ++tz)
                    for (int u = 0; u < 4; ++u) {
                        slot_of[f][tt][tz][u] = -1;
                        int tx, ty;
                        if (f < 2) { tx = (f == 0) ? 0 : 3; ty = u; if (((q + tx + ty + tz + tt) & 1) != 0) continue; }
                        else { if (u >= 2) continue; ty = (f == 2) ? 0 : 3; tx = 2 * u + ((q + ty + tz + tt) & 1); }
                        const int pos = ty ^ tz;
                        int region, slot;
                        if (f < 2) {
                            const int b = 2 * pos + f;                       // +x even groups, -x odd groups
                            const int s64 = b + 8 * cnt[f][b]++;
                            region = 10 + (s64 >> 5); slot = s64 & 31;
                        } else {
                            const int b = 2 * pos + (tx >> 1);
                            slot = b + 8 * cnt[f][b]++;
                            region = (f == 2) ? 8 : 9;
                        }
                        slot_of[f][tt][tz][u] = region * K * 32 + slot;
                        const int i = nface[f]++;
                        t.gsrc[(p * 4 + f) * 32 + i] = (uint8_t)lane_of(tx, ty, tz, tt);
                        t.gdst[(p * 4 + f) * 32 + i] = (uint16_t)(region * K * 32 + slot);
                    }
        // ---- every output site's 8 neighbours
        for (int tt = 0; tt < 4; ++tt)
            for (int tz = 0; tz < 4; ++tz)
                for (int ty = 0; ty < 4; ++ty)
                    for (int txh = 0; txh < 2; ++txh) {
                        const int tx = 2 * txh + ((p + ty + tz + tt) & 1);
                        const int lane = lane_of(tx, ty, tz, tt);
                        for (int leg = 0; leg < 8; ++leg) {
                            const int mu = leg >> 1;
                            int y[4] = {tx, ty, tz, tt};
                            y[mu] += (leg & 1) ? -1 : +1;
                            int o;
                            if (y[mu] >= 0 && y[mu] < 4) {
                                o = y[3] * K * 32 + (lane_of(y[0], y[1], y[2], y[3]) & 31);          // own slab y[3]
                            } else {
                                const int up = (y[mu] >= 4);
                                y[mu] = (y[mu] + 4) & 3;
                                if (mu == 3)      o = (up ? 4 : 5) * K * 32 + (lane_of(y[0], y[1], y[2], 0) & 31);   // t face: one slab
                                else if (mu == 2) o = (up ? 6 : 7) * K * 32 + y[3] * 8 + (y[1] ^ y[2]) * 2 + (y[0] >> 1);  // z face: 8 lanes x tt
                                else if (mu == 1) o = slot_of[up ? 2 : 3][y[3]][y[2]][y[0] >> 1];
                                else              o = slot_of[up ? 0 : 1][y[3]][y[2]][y[1]];
                            }
                            t.off[(p * 8 + leg) * TSV + lane] = (uint16_t)o;
                        }
                    }
    }
    return t;
}

// Tile traversal.  The persistent CTAs take order[blockIdx], order[blockIdx + grid], ...: at any time the tiles in
// flight are about one grid-sized run of `order`.  The runs are compact 4-D blobs of B[0] x B[1] x B[2] x B[3] tiles
// (faces between tiles of one blob are read by two CTAs at about the same time: L2 hits), and the blobs follow each
// other in a boustrophedon path (axes[0] fastest), so that a blob's faces towards the previous blob are still in L2.
// code = B0 B1 B2 B3 as decimal digits (0 = full extent), axes = fastest-first axis digits of the blob path
// (DESIGN.md §5).  Default: 8x8x2x1 blobs swept along t, then z.
std::vector<uint32_t> build_order(const Geom& g, int code, int axes_code) {
    int B[4], ax[4];
    if (code <= 0) { code = 21; axes_code = 3210; }   // 0 0 2 1
    int digs[4] = {(code / 1000) % 10, (code / 100) % 10, (code / 10) % 10, code % 10};
    for (int mu = 0; mu < 4; ++mu) {
        B[mu] = digs[mu] <= 0 ? g.NT[mu] : std::min(digs[mu], g.NT[mu]);
        while (g.NT[mu] % B[mu] != 0) --B[mu];
    }
    int ad[4] = {(axes_code / 1000) % 10, (axes_code / 100) % 10, (axes_code / 10) % 10, axes_code % 10};
    bool seen[4] = {false, false, false, false};
    int na = 0;
    for (int i = 0; i < 4; ++i)
        if (ad[i] >= 0 && ad[i] < 4 && !seen[ad[i]]) { ax[na++] = ad[i]; seen[ad[i]] = true; }
    for (int mu = 3; mu >= 0; --mu)
        if (!seen[mu]) { ax[na++] = mu; seen[mu] = true; }
    int NB[4];
    for (int mu = 0; mu < 4; ++mu) NB[mu] = g.NT[mu] / B[mu];
    std::vector<uint32_t> o;
    o.reserve(g.ntiles);
    const int nblobs = NB[0] * NB[1] * NB[2] * NB[3];
    auto blob_coords = [&](int ib, int bc[4]) {
        // mixed-radix digits of ib (ax[0] fastest), reflected when the sum of the higher digits is odd
        int d[4], r = ib;
        for (int i = 0; i < 4; ++i) { d[i] = r % NB[ax[i]]; r /= NB[ax[i]]; }
        for (int i = 3; i >= 0; --i) {
            int hi = 0;
            for (int j = i + 1; j < 4; ++j) hi += d[j];
            bc[ax[i]] = (hi & 1) ? NB[ax[i]] - 1 - d[i] : d[i];
        }
    };
    for (int ib = 0; ib < nblobs; ++ib) {
        int bc[4];
        blob_coords(ib, bc);
        for (int t = 0; t < B[3]; ++t)
            for (int z = 0; z < B[2]; ++z)
                for (int y = 0; y < B[1]; ++y)
                    for (int x = 0; x < B[0]; ++x) {
                        const int c[4] = {bc[0] * B[0] + x, bc[1] * B[1] + y, bc[2] * B[2] + z, bc[3] * B[3] + t};
                        o.push_back((uint32_t)tile_index(g, c));
                    }
    }
    return o;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
        cudaGetLastError();
    }
    return fn;
}

}  // namespace

struct TmaState {
    uint16_t* off = nullptr;      // device [2][8][128]
    uint8_t* xsrc = nullptr;      // device [2][2][32]   (fp32 path)
    uint16_t* xdst = nullptr;     // device [2][2][32]   (fp32 path)
    uint8_t* gsrc = nullptr;      // device [2][4][32]   (fp64 path)
    uint16_t* gdst = nullptr;     // device [2][4][32]   (fp64 path)
    uint32_t* order = nullptr;    // device [ntiles]
    int* counters = nullptr;      // device [3]: next position in `order`, CTAs done, round arrivals (self-resetting, see the kernel)
    int K_built = 0;
    int num_sms = 0;
    struct Maps { const void* ptr; int prec; int Ls; CUtensorMap m[3]; };
    std::vector<Maps> cache;      // small LRU of tensor maps per input pointer
};

void tma_state_free(dwf_ctx* c) {
    TmaState* s = (TmaState*)c->tma;
    if (!s) return;
    if (s->off) cudaFree(s->off);
    if (s->xsrc) cudaFree(s->xsrc);
    if (s->xdst) cudaFree(s->xdst);
    if (s->gsrc) cudaFree(s->gsrc);
    if (s->gdst) cudaFree(s->gdst);
    if (s->order) cudaFree(s->order);
    if (s->counters) cudaFree(s->counters);
    delete s;
    c->tma = nullptr;
}

// built at dwf_set_gauge (geometry is frozen there); returns DWF_OK with c->tma == nullptr when the tile shape
// or the driver has no TMA path
dwf_status tma_state_build(dwf_ctx* c) {
    tma_state_free(c);
    const Geom& g = c->g;
    for (int mu = 0; mu < 4; ++mu)
        if (g.T[mu] != 4) return DWF_OK;
    if (!encode_fn()) return DWF_OK;
    TmaState* s = new TmaState();
    c->tma = s;            // tma_state_free releases a half-built state; published for launches only on success (below)
    dwf_status st = [&]() -> dwf_status {
        cudaDeviceGetAttribute(&s->num_sms, cudaDevAttrMultiProcessorCount, c->device);
        // fp64 tables first (K = 12, XOR-rotated lane order), fp32 second (K = 6, plain order)
        TmaTables t64 = build_tma_tables_swz(12), t32 = build_tma_tables_plain(6);
        std::vector<uint16_t> off(t64.off);
        off.insert(off.end(), t32.off.begin(), t32.off.end());
        const std::vector<uint16_t>& gdst = t64.gdst;
        std::vector<uint32_t> order = build_order(g, 0, 0);
        DWF_CUDA_CHECK(c, cudaMalloc(&s->off, off.size() * sizeof(uint16_t)));
        DWF_CUDA_CHECK(c, cudaMalloc(&s->xsrc, t32.xsrc.size()));
        DWF_CUDA_CHECK(c, cudaMalloc(&s->xdst, t32.xdst.size() * sizeof(uint16_t)));
        DWF_CUDA_CHECK(c, cudaMalloc(&s->gsrc, t64.gsrc.size()));
        DWF_CUDA_CHECK(c, cudaMalloc(&s->gdst, gdst.size() * sizeof(uint16_t)));
        DWF_CUDA_CHECK(c, cudaMalloc(&s->order, order.size() * sizeof(uint32_t)));
        DWF_CUDA_CHECK(c, cudaMemcpy(s->off, off.data(), off.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMemcpy(s->xsrc, t32.xsrc.data(), t32.xsrc.size(), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMemcpy(s->xdst, t32.xdst.data(), t32.xdst.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMemcpy(s->gsrc, t64.gsrc.data(), t64.gsrc.size(), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMemcpy(s->gdst, gdst.data(), gdst.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMemcpy(s->order, order.data(), order.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
        DWF_CUDA_CHECK(c, cudaMalloc(&s->counters, 4 * sizeof(int)));
        DWF_CUDA_CHECK(c, cudaMemset(s->counters, 0, 4 * sizeof(int)));
        return DWF_OK;
    }();
    if (st != DWF_OK) tma_state_free(c);      // never leave half-built tables behind: later launches would dereference them
    return st;
}

// three tensor maps over one native half field: [0] t-slabs (512-byte rows), [1] z faces (128-byte rows),
// [2] y faces (32-byte rows).  A native half field is nrows = ntiles*Ls*K rows of 2048 bytes (one (tile,s,k) each).
static dwf_status get_maps(dwf_ctx* c, const void* in, int prec, const CUtensorMap** out) {
    TmaState* s = (TmaState*)c->tma;
    const int LsT = c->g.Ls * c->nrhs_cur;                // batched fields: one long fifth dimension
    for (size_t i = 0; i < s->cache.size(); ++i)
        if (s->cache[i].ptr == in && s->cache[i].prec == prec && s->cache[i].Ls == LsT) {
            if (i != 0) std::swap(s->cache[i], s->cache[0]);
            *out = s->cache[0].m;
            return DWF_OK;
        }
    const Geom& g = c->g;
    const int K = (prec == DWF_F64) ? 12 : 6;
    const int epv = (prec == DWF_F64) ? 2 : 4;             // elements per 16-byte vector
    const cuuint64_t nrows = (cuuint64_t)g.ntiles * LsT * K;
    const CUtensorMapDataType dt = (prec == DWF_F64) ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    TmaState::Maps m;
    m.ptr = in; m.prec = prec; m.Ls = LsT;
    EncodeTiledFn enc = encode_fn();
    const cuuint32_t ones[4] = {1, 1, 1, 1};
    CUresult r;
    {   // slabs: (32 lanes, tt, row)
        const cuuint64_t dims[3] = {(cuuint64_t)32 * epv, 4, nrows};
        const cuuint64_t strides[2] = {512, 2048};
        const cuuint32_t box[3] = {(cuuint32_t)32 * epv, 1, (cuuint32_t)K};
        r = enc(&m.m[0], dt, 3, const_cast<void*>(in), dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { c->err = "cuTensorMapEncodeTiled(slab) failed"; return DWF_ECUDA; }
    }
    {   // z faces: (8 lanes = ty,txh; tz; tt; row)
        const cuuint64_t dims[4] = {(cuuint64_t)8 * epv, 4, 4, nrows};
        const cuuint64_t strides[3] = {128, 512, 2048};
        const cuuint32_t box[4] = {(cuuint32_t)8 * epv, 1, 4, (cuuint32_t)K};
        r = enc(&m.m[1], dt, 4, const_cast<void*>(in), dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { c->err = "cuTensorMapEncodeTiled(z) failed"; return DWF_ECUDA; }
    }
    {   // y faces: (2 lanes = txh; ty; (tz,tt); row)
        const cuuint64_t dims[4] = {(cuuint64_t)2 * epv, 4, 16, nrows};
        const cuuint64_t strides[3] = {32, 128, 2048};
        const cuuint32_t box[4] = {(cuuint32_t)2 * epv, 1, 16, (cuuint32_t)K};
        r = enc(&m.m[2], dt, 4, const_cast<void*>(in), dims, strides, box, ones, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { c->err = "cuTensorMapEncodeTiled(y) failed"; return DWF_ECUDA; }
    }
    s->cache.insert(s->cache.begin(), m);
    if (s->cache.size() > 32) s->cache.pop_back();
    *out = s->cache[0].m;
    return DWF_OK;
}

// ------------------------------------------------------------------------------------------ device helpers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void cp_async16_tma(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint32_t bar) {
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}
__device__ __forceinline__ void l2_prefetch(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void l2_prefetch_bulk(const void* p, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
template <int N> __device__ __forceinline__ void reg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N> __device__ __forceinline__ void reg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }

__device__ __forceinline__ float4 lds_v(const float4*, uint32_t a) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ double2 lds_v(const double2*, uint32_t a) {
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ void stcs_v(float4* p, const float4& v) { __stcs(p, v); }
__device__ __forceinline__ void stcs_v(double2* p, const double2& v) { __stcs(p, v); }

// global loads the compiler may not sink below the slice's shared-memory loads (both are volatile asm, kept in order)
__device__ __forceinline__ float4 ldg_early(const float4* p) {
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ double2 ldg_early(const double2* p) {
    double2 v;
    asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ void pin_reg(float& v) { asm volatile("" : "+f"(v)); }
__device__ __forceinline__ void pin_reg(double& v) { asm volatile("" : "+d"(v)); }
__device__ __forceinline__ float shfl16(float v) { return __shfl_xor_sync(0xffffffffu, v, 16); }
__device__ __forceinline__ double shfl16(double v) { return __shfl_xor_sync(0xffffffffu, v, 16); }

// h = upper two rows of (1 + s*gamma_MU) psi, s = +-1 at run time (FMA form)
template <typename R, int MU>
__device__ __forceinline__ void proj_s(const R (&psi)[24], R s, R (&h)[12]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int p0 = 2 * c, p1 = 6 + 2 * c, p2 = 12 + 2 * c, p3 = 18 + 2 * c;
        const int h0 = 2 * c, h1 = 6 + 2 * c;
        if (MU == 0) {
            h[h0] = psi[p0] - s * psi[p3 + 1]; h[h0 + 1] = psi[p0 + 1] + s * psi[p3];
            h[h1] = psi[p1] - s * psi[p2 + 1]; h[h1 + 1] = psi[p1 + 1] + s * psi[p2];
        } else if (MU == 1) {
            h[h0] = psi[p0] - s * psi[p3]; h[h0 + 1] = psi[p0 + 1] - s * psi[p3 + 1];
            h[h1] = psi[p1] + s * psi[p2]; h[h1 + 1] = psi[p1 + 1] + s * psi[p2 + 1];
        } else if (MU == 2) {
            h[h0] = psi[p0] - s * psi[p2 + 1]; h[h0 + 1] = psi[p0 + 1] + s * psi[p2];
            h[h1] = psi[p1] + s * psi[p3 + 1]; h[h1 + 1] = psi[p1 + 1] - s * psi[p3];
        } else {
            h[h0] = psi[p0] + s * psi[p2]; h[h0 + 1] = psi[p0 + 1] + s * psi[p2 + 1];
            h[h1] = psi[p1] + s * psi[p3]; h[h1 + 1] = psi[p1 + 1] + s * psi[p3 + 1];
        }
    }
}

// acc (+)= reconstruct((1 + s*gamma_MU) from g); FIRST: assign instead of accumulate
template <typename R, int MU, bool FIRST>
__device__ __forceinline__ void recon_s(const R (&g)[12], R s, R (&acc)[24]) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const int g0 = 2 * c, g1 = 6 + 2 * c;
        const int a0 = 2 * c, a1 = 6 + 2 * c, a2 = 12 + 2 * c, a3 = 18 + 2 * c;
        R l2r, l2i, l3r, l3i;   // lower rows
        if (MU == 0)      { l2r = s * g[g1 + 1]; l2i = -s * g[g1]; l3r = s * g[g0 + 1]; l3i = -s * g[g0]; }
        else if (MU == 1) { l2r = s * g[g1]; l2i = s * g[g1 + 1]; l3r = -s * g[g0]; l3i = -s * g[g0 + 1]; }
        else if (MU == 2) { l2r = s * g[g0 + 1]; l2i = -s * g[g0]; l3r = -s * g[g1 + 1]; l3i = s * g[g1]; }
        else              { l2r = s * g[g0]; l2i = s * g[g0 + 1]; l3r = s * g[g1]; l3i = s * g[g1 + 1]; }
        if (FIRST) {
            acc[a0] = g[g0]; acc[a0 + 1] = g[g0 + 1]; acc[a1] = g[g1]; acc[a1 + 1] = g[g1 + 1];
            acc[a2] = l2r; acc[a2 + 1] = l2i; acc[a3] = l3r; acc[a3 + 1] = l3i;
        } else {
            acc[a0] += g[g0]; acc[a0 + 1] += g[g0 + 1]; acc[a1] += g[g1]; acc[a1 + 1] += g[g1 + 1];
            if (MU == 0)      { acc[a2] += s * g[g1 + 1]; acc[a2 + 1] -= s * g[g1]; acc[a3] += s * g[g0 + 1]; acc[a3 + 1] -= s * g[g0]; }
            else if (MU == 1) { acc[a2] += s * g[g1]; acc[a2 + 1] += s * g[g1 + 1]; acc[a3] -= s * g[g0]; acc[a3 + 1] -= s * g[g0 + 1]; }
            else if (MU == 2) { acc[a2] += s * g[g0 + 1]; acc[a2 + 1] -= s * g[g0]; acc[a3] -= s * g[g1 + 1]; acc[a3 + 1] += s * g[g1]; }
            else              { acc[a2] += s * g[g0]; acc[a2 + 1] += s * g[g0 + 1]; acc[a3] += s * g[g1]; acc[a3 + 1] += s * g[g1 + 1]; }
        }
    }
}


// ------------------------------------------------------------------------------------------ fused epilogue
// The last step of Mpc rides on the Dhop kernel:  out_s = Mee xin_s + scale * (Dhop in)_s  with |out|^2 (EPI_FINAL).
// Mee = bee - cee Q is bidiagonal in s (reading C5): P+ components take xin_{s-1}, P- components xin_{s+1}, with the
// -mf wall; the hopping term enters pointwise, so nothing but the slice being written has to stay on chip.
// (The column-global operators -- Mee^-1 and the A^dag that follows a daggered Dhop -- stay in the column kernels of
// dwf_fived.cu: an Ls column of one tile does not fit in registers or shared memory next to the staging ring, and a
// round trip through a global scratch tile costs a DRAM write-back on this L2.)
struct EpiArgs {
    int mode;              // EPI_NONE or EPI_FINAL
    const void* xin;       // the field Mee acts on (output parity)
    double* partials;      // partial sums of |out|^2, one per (system, tile): partials[rhs * ntiles + tile]; null: none
    double bee, mcee, mf, scale;     // Mee = bee + mcee Q
    int Ls0;               // physical Ls: a batched field has g.Ls = N * Ls0 slices per tile, walls at s mod Ls0 = 0, Ls0 - 1
};

__device__ __forceinline__ float4 vmul(float a, const float4& x) { return make_float4(a * x.x, a * x.y, a * x.z, a * x.w); }
__device__ __forceinline__ double2 vmul(double a, const double2& x) { return make_double2(a * x.x, a * x.y); }
__device__ __forceinline__ float4 vfma(float a, const float4& x, const float4& y) {
    return make_float4(fmaf(a, x.x, y.x), fmaf(a, x.y, y.y), fmaf(a, x.z, y.z), fmaf(a, x.w, y.w));
}
__device__ __forceinline__ double2 vfma(double a, const double2& x, const double2& y) {
    return make_double2(fma(a, x.x, y.x), fma(a, x.y, y.y));
}
__device__ __forceinline__ double vnorm2(const float4& a) {
    return (double)a.x * a.x + (double)a.y * a.y + (double)a.z * a.z + (double)a.w * a.w;
}
__device__ __forceinline__ double vnorm2(const double2& a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ float4 ldcs_v(const float4* p) { return __ldcs(p); }
__device__ __forceinline__ double2 ldcs_v(const double2* p) { return __ldcs(p); }

struct TmaArgs {
    Geom g;
    const void* in;
    void* out;
    const void* W;
    const uint16_t* off;      // [8][128]   (this output parity, this precision)
    const uint8_t* xsrc;      // [2][32]    fp32: x-face source lanes (this output parity)
    const uint16_t* xdst;     // [2][32]    fp32: ... and stage offsets
    const uint8_t* gsrc;      // [4][32]    fp64: gathered faces +x, -x, +y, -y: source lanes (this output parity)
    const uint16_t* gdst;     // [4][32]    ... and stage offsets (this output parity, this precision)
    const uint32_t* order;    // [ntiles]
    int* counters;            // [3] queue / done / round-arrival counters
    EpiArgs epi;
    int mode;                 // 0: static round-robin, 1: global in-order queue
    int dagger;
};


template <typename R, int TPS, int NG, int NST, int MINB, int EPI>
__global__ void __launch_bounds__(128 + 128 * TPS, MINB)
dhop_tma_kernel(const TmaArgs a, const __grid_constant__ CUtensorMap map_slab, const __grid_constant__ CUtensorMap map_z,
                const __grid_constant__ CUtensorMap map_y) {
    using V = typename VT<R>::V;
    constexpr int K = VT<R>::K, VW = VT<R>::VW;
    constexpr int KG = (NG + VW - 1) / VW;
    constexpr int LPT = 8 / TPS;
    constexpr int NCW = 4 * TPS;                       // consumer warps
    constexpr uint32_t REGION_BYTES = K * 512;
    constexpr uint32_t STAGE_BYTES = NREG * REGION_BYTES;
    // setmaxnreg: the pool is the launch allocation, so (launch - PROD) x 128 must cover (CONS - launch) x consumers, or the
    // consumers' setmaxnreg.inc blocks for ever.  fp64 (168 at launch, 256 consumers): 32 / 232; fp32 (128, 128): 24 / 232
    constexpr int REG_PROD = (TPS == 2) ? 32 : 24;
    constexpr int REG_CONS = 232;

    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[2 * NST];   // full[NST], empty[NST]
    __shared__ double wsum[4 * TPS];      // per-(system, tile) |.|^2 partials of the consumer warps (fused epilogue)
    __shared__ int next_of[4];     // slot j & 3, written before slice 0 of this CTA's j-th tile: the tile it takes after it (-1: none)

    const Geom& g = a.g;
    const int Ls = g.Ls;
    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;
    const uint32_t stage0 = smem_u32(smem_raw);
    const uint32_t bar0 = smem_u32(bars);
    const int ntiles = g.ntiles;

    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < NST; ++i) {
            mbar_init(bar0 + 8 * i, 1 + 32);             // full: producer's expect_tx arrive + 32 cp.async arrivals
            mbar_init(bar0 + 8 * (NST + i), NCW);        // empty: one arrival per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (warp < 4) {
        // ================================================================================== PRODUCER
        reg_dec<REG_PROD>();
        if (warp != 0) return;
        const V* __restrict__ in = reinterpret_cast<const V*>(a.in);
        // gathered faces: this lane's source lane in the neighbour tile and its slot in the stage.
        // fp64 (GATHER_Y): +x, -x, +y, -y faces into the conflict-free slots of build_tma_tables_swz;
        // fp32: +x, -x faces interleaved over regions 10, 11, the y faces come by TMA (build_tma_tables_plain)
        constexpr bool GATHER_Y = (TPS == 2);
        const uint32_t gs0 = GATHER_Y ? a.gsrc[lane] : a.xsrc[lane], gs1 = GATHER_Y ? a.gsrc[32 + lane] : a.xsrc[32 + lane];
        const uint32_t gd0 = (uint32_t)(GATHER_Y ? a.gdst[lane] : a.xdst[lane]) * 16u;
        const uint32_t gd1 = (uint32_t)(GATHER_Y ? a.gdst[32 + lane] : a.xdst[32 + lane]) * 16u;
        const uint32_t gs2 = GATHER_Y ? a.gsrc[64 + lane] : 0, gs3 = GATHER_Y ? a.gsrc[96 + lane] : 0;
        const uint32_t gd2 = GATHER_Y ? (uint32_t)a.gdst[64 + lane] * 16u : 0, gd3 = GATHER_Y ? (uint32_t)a.gdst[96 + lane] * 16u : 0;
        constexpr int NTMA = GATHER_Y ? 8 : 10;      // regions written by TMA boxes
        const uint32_t tile_vecs = (uint32_t)Ls * K * TSV;
        uint32_t n = 0, j = 0;
        int it = blockIdx.x;
        while (it < ntiles) {
            // next position in `order`: static round-robin, or the global in-order queue (tiles start in `order`
            // sequence whatever the CTAs' speeds)
            int it_next = it + gridDim.x;
            if (a.mode == 1) {
                int v = 0;
                if (lane == 0) v = atomicAdd(a.counters, 1) + (int)gridDim.x;
                it_next = __shfl_sync(0xffffffffu, v, 0);
            }
            const int tile = (int)a.order[it];
            const int tile_next = (it_next < ntiles) ? (int)a.order[it_next] : -1;
            int tc[4];
            tile_coords(g, tile, tc);
            int nt[8];
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {
                int nc[4] = {tc[0], tc[1], tc[2], tc[3]};
                nc[mu] = (tc[mu] + 1 == g.NT[mu]) ? 0 : tc[mu] + 1;
                nt[2 * mu] = tile_index(g, nc);
                nc[mu] = (tc[mu] == 0) ? g.NT[mu] - 1 : tc[mu] - 1;
                nt[2 * mu + 1] = tile_index(g, nc);
            }
            if (lane == 0) next_of[j & 3] = tile_next;       // published by the release-arrive on slice 0's `full` barrier
            ++j;
            // vector indices (< 2^31, checked at dwf_create) of this lane's face sources at s = 0
            const uint32_t i0 = (uint32_t)nt[0] * tile_vecs + gs0, i1 = (uint32_t)nt[1] * tile_vecs + gs1;
            const uint32_t i2 = (uint32_t)nt[2] * tile_vecs + gs2, i3 = (uint32_t)nt[3] * tile_vecs + gs3;
            for (int s = 0; s < Ls; ++s, ++n) {
                const uint32_t st = n % NST, ph = (n / NST) & 1;
                const uint32_t full = bar0 + 8 * st, empty = bar0 + 8 * (NST + st);
                const uint32_t base = stage0 + st * STAGE_BYTES;
                mbar_wait(empty, ph ^ 1);
                if (lane == 0) {
                    // next tile's links -> L2, issued with this tile's last slice: the consumers want them NST slices
                    // later (issued a whole tile ahead they were evicted again before use and fetched twice)
                    if (s == Ls - 1 && tile_next >= 0)
                        l2_prefetch_bulk(reinterpret_cast<const V*>(a.W) + (size_t)tile_next * 8 * KG * TSV, 8 * KG * TSV * 16);
                    mbar_arrive_expect_tx(full, NTMA * REGION_BYTES);
                    const int row_own = (tile * Ls + s) * K;
#pragma unroll
                    for (int tt = 0; tt < 4; ++tt) tma_load_3d(base + tt * REGION_BYTES, &map_slab, 0, tt, row_own, full);
                    tma_load_3d(base + 4 * REGION_BYTES, &map_slab, 0, 0, (nt[6] * Ls + s) * K, full);
                    tma_load_3d(base + 5 * REGION_BYTES, &map_slab, 0, 3, (nt[7] * Ls + s) * K, full);
                    tma_load_4d(base + 6 * REGION_BYTES, &map_z, 0, 0, 0, (nt[4] * Ls + s) * K, full);
                    tma_load_4d(base + 7 * REGION_BYTES, &map_z, 0, 3, 0, (nt[5] * Ls + s) * K, full);
                    if (!GATHER_Y) {
                        tma_load_4d(base + 8 * REGION_BYTES, &map_y, 0, 0, 0, (nt[2] * Ls + s) * K, full);
                        tma_load_4d(base + 9 * REGION_BYTES, &map_y, 0, 3, 0, (nt[3] * Ls + s) * K, full);
                    }
                }
                const V* src = in + (size_t)s * (K * TSV);
#pragma unroll
                for (int k = 0; k < K; ++k) {
                    cp_async16_tma(base + gd0 + k * 512, src + i0 + k * TSV);
                    cp_async16_tma(base + gd1 + k * 512, src + i1 + k * TSV);
                    if (GATHER_Y) {
                        cp_async16_tma(base + gd2 + k * 512, src + i2 + k * TSV);
                        cp_async16_tma(base + gd3 + k * 512, src + i3 + k * TSV);
                    }
                }
                cp_async_mbar_arrive_noinc(full);
            }
            it = it_next;
        }
        if (a.mode != 0 && lane == 0) {          // the last CTA out re-arms the counters for the next launch
            __threadfence();
            if (atomicAdd(a.counters + 1, 1) == (int)gridDim.x - 1) {
                atomicExch(a.counters, 0);
                atomicExch(a.counters + 1, 0);
                atomicExch(a.counters + 2, 0);
            }
        }
        return;
    }

    // ====================================================================================== CONSUMERS
    reg_inc<REG_CONS>();
    const int ctid = tid - 128;
    const int cw = ctid >> 5;
    int sub, site;
    if (TPS == 1) { sub = 0; site = ctid; }
    else { sub = lane >> 4; site = cw * 16 + (lane & 15); }

    uint32_t myoff[LPT];
#pragma unroll
    for (int j = 0; j < LPT; ++j) {
        const int leg = (TPS == 1) ? j : 2 * j + sub;
        myoff[j] = (uint32_t)a.off[leg * TSV + site] * 16u;
    }
    const int tt = site >> 5;
    const R dsgn = a.dagger ? (R)-1 : (R)1;
    uint32_t n = 0, j = 0;
    double nrm = 0.0;
    int tile = (int)a.order[blockIdx.x];
    while (tile >= 0) {
        int tile_next = -1;
        const int tct = tile / (g.NT[0] * g.NT[1] * g.NT[2]);
        const int tglob = tct * 4 + tt;
        // ---- links to registers (once per tile): rows 0,1 (+ row 2 rebuilt), antiperiodic sign folded in.
        // REMAT (fp64 kernel with the fused epilogue): only rows 0, 1 stay in registers and row 2 is rebuilt in every slice
        // (+18 % FP64 instructions) -- the 48 registers this frees hold the epilogue's 12 global loads, issued at the top of
        // the slice instead of at its end where nothing hid their latency (long-scoreboard stalls 3.2 per issue before)
        constexpr bool REMAT = (EPI != 0) && (sizeof(R) == 8) && (NG == 12);
        R u[LPT][18];
        R tsgn = (R)1;                  // REMAT: antiperiodic sign of this lane's t leg, applied to the rebuilt row
        {
            const V* __restrict__ Wt = reinterpret_cast<const V*>(a.W) + (size_t)tile * 8 * KG * TSV + site;
#pragma unroll
            for (int j = 0; j < LPT; ++j) {
                const int leg = (TPS == 1) ? j : 2 * j + sub;
                load_link<R, NG>(Wt + (size_t)leg * KG * TSV, TSV, u[j]);
                const int mu = (TPS == 1) ? (j >> 1) : j;
                if (mu == 3 && g.antiperiodic_t) {
                    const int dir = (TPS == 1) ? (j & 1) : sub;
                    const bool flip = dir ? (tglob == 0) : (tglob == g.L[3] - 1);
                    if (flip) {
#pragma unroll
                        for (int i = 0; i < 18; ++i) u[j][i] = -u[j][i];
                        tsgn = (R)-1;
                    }
                }
                // fp32, plain kernel: the rebuilt third row stays in registers for the whole tile: without this the compiler,
                // short of registers, recomputes it from rows 0, 1 in every slice (+19 % FP instructions in the s loop:
                // 1032 -> 870; the fp64 loop has no such recomputation).  Not in the fused kernel: there the registers the
                // recomputation frees let the epilogue's global loads issue early (414 us vs 529 us with the rows pinned).
                if (NG == 12 && sizeof(R) == 4 && EPI == 0) {
#pragma unroll
                    for (int i = 12; i < 18; ++i) pin_reg(u[j][i]);
                }
            }
        }
        V* __restrict__ outp = reinterpret_cast<V*>(a.out) + (size_t)tile * Ls * K * TSV + site;
        const V* __restrict__ xin_t = reinterpret_cast<const V*>(a.epi.xin) + (size_t)tile * Ls * K * TSV + site;
        // fused epilogue on a batched field: sl = slice within its system (0 .. Ls0-1); s - sl = first slice of that system
        int sl = 0;
        for (int s = 0; s < Ls; ++s, ++n) {
            const uint32_t st = n % NST, ph = (n / NST) & 1;
            const uint32_t base = stage0 + st * STAGE_BYTES;
            mbar_wait(bar0 + 8 * st, ph);
            if (s == 0) tile_next = *(volatile int*)&next_of[j & 3];
            if constexpr (EPI != 0) {
                // the epilogue's xin rows -> L2 one slice ahead (a system's slice 0 also fetches itself and the wall slice)
                const V* xk = xin_t + ((TPS == 1) ? 0 : sub * (K / 2)) * TSV;
                if (s + 1 < Ls) {
#pragma unroll
                    for (int k = 0; k < 6; ++k) l2_prefetch(xk + (size_t)(s + 1) * (K * TSV) + k * TSV);
                }
                if (sl == 0) {
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        l2_prefetch(xk + (size_t)s * (K * TSV) + k * TSV);
                        l2_prefetch(xk + (size_t)(s + a.epi.Ls0 - 1) * (K * TSV) + k * TSV);
                    }
                }
            }
            // REMAT: this lane's epilogue operands (its chirality half of xin_s and of xin_{s-1} / xin_{s+1}) -> registers,
            // requested here; ptxas places the loads as early as its register budget allows (in the exchange phase, well
            // before their use; loading them one whole slice ahead spilled and was slower: 988 us vs 920 us)
            V xcv[K / 2], xnv[K / 2];
            if (REMAT && EPI != 0) {
                const int Ls0e = a.epi.Ls0;
                const V* xs_e = xin_t + (size_t)s * (K * TSV) + (sub ? K / 2 : 0) * TSV;
                const int sn = sub ? ((sl + 1 < Ls0e) ? s + 1 : s + 1 - Ls0e) : ((sl > 0) ? s - 1 : s + Ls0e - 1);
                const V* xn_e = xin_t + (size_t)sn * (K * TSV) + (sub ? K / 2 : 0) * TSV;
#pragma unroll
                for (int k = 0; k < K / 2; ++k) { xcv[k] = ldg_early(xs_e + k * TSV); xnv[k] = ldg_early(xn_e + k * TSV); }
            }
            R acc[24];
#pragma unroll
            for (int j = 0; j < LPT; ++j) {
                const int mu = (TPS == 1) ? (j >> 1) : j;
                const int dir = (TPS == 1) ? (j & 1) : sub;
                const R sg = (dir ? (R)1 : (R)-1) * dsgn;     // forward leg: (1 - gamma), backward: (1 + gamma)
                R psi[24], h[12], gg[12];
                const uint32_t p = base + myoff[j];
#pragma unroll
                for (int k = 0; k < K; ++k) unpackv(lds_v((const V*)nullptr, p + k * 512), psi + k * VW);
                if (REMAT) {
                    pin_reg(u[j][0]);                  // opaque: keeps the rebuild inside the slice loop
                    third_row<R>(u[j]);
                    if (mu == 3) {
#pragma unroll
                        for (int i = 12; i < 18; ++i) u[j][i] *= tsgn;
                    }
                }
                if (j == 0) { proj_s<R, 0>(psi, sg, h); su3_mul<R>(u[j], h, gg); recon_s<R, 0, true>(gg, sg, acc); }
                else if (mu == 0) { proj_s<R, 0>(psi, sg, h); su3_mul<R>(u[j], h, gg); recon_s<R, 0, false>(gg, sg, acc); }
                else if (mu == 1) { proj_s<R, 1>(psi, sg, h); su3_mul<R>(u[j], h, gg); recon_s<R, 1, false>(gg, sg, acc); }
                else if (mu == 2) { proj_s<R, 2>(psi, sg, h); su3_mul<R>(u[j], h, gg); recon_s<R, 2, false>(gg, sg, acc); }
                else { proj_s<R, 3>(psi, sg, h); su3_mul<R>(u[j], h, gg); recon_s<R, 3, false>(gg, sg, acc); }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar0 + 8 * (NST + st));      // stage released
            V* o = outp + (size_t)s * (K * TSV);
            // EPI: out_s = bee xin_s + mcee (Q xin)_s + scale D_s, |out|^2 summed (Mee xin - 1/4 Dhop ..., reading C6)
            const R e_bee = (R)a.epi.bee, e_scale = (R)a.epi.scale;
            const int Ls0 = (EPI != 0) ? a.epi.Ls0 : Ls;
            const R e_wm = (R)((sl > 0) ? a.epi.mcee : -a.epi.mf * a.epi.mcee);            // P+ : xin_{s-1}
            const R e_wp = (R)((sl + 1 < Ls0) ? a.epi.mcee : -a.epi.mf * a.epi.mcee);      // P- : xin_{s+1}
            const V* xs = xin_t + (size_t)s * (K * TSV);
            const V* xm = xin_t + (size_t)((sl > 0) ? s - 1 : s + Ls0 - 1) * (K * TSV);
            const V* xp = xin_t + (size_t)((sl + 1 < Ls0) ? s + 1 : s + 1 - Ls0) * (K * TSV);
            if (TPS == 1) {
                if constexpr (EPI != 0) {
#pragma unroll
                    for (int k = 0; k < K; ++k) {
                        const V xc = ldg_v(xs + k * TSV);
                        const V xn = ldg_v(((k < K / 2) ? xm : xp) + k * TSV);
                        const V ov = vfma(e_scale, packv(acc + k * VW), vfma((k < K / 2) ? e_wm : e_wp, xn, vmul(e_bee, xc)));
                        nrm += vnorm2(ov);
                        stcs_v(o + k * TSV, ov);
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < K; ++k) stcs_v(o + k * TSV, packv(acc + k * VW));
                }
            } else {
                // lane pair (l, l^16): each keeps one chirality half of the 24 sums, sends the other
                R mine[12];
#pragma unroll
                for (int i = 0; i < 12; ++i) {
                    const R send = sub ? acc[i] : acc[12 + i];
                    const R keep = sub ? acc[12 + i] : acc[i];
                    mine[i] = keep + shfl16(send);
                }
                const int k0 = sub ? (K / 2) : 0;
                V* o2 = o + k0 * TSV;
                if constexpr (EPI != 0) {
                    const V* xc_p = xs + k0 * TSV;
                    const V* xn_p = (sub ? xp : xm) + k0 * TSV;
                    const R w = sub ? e_wp : e_wm;
#pragma unroll
                    for (int k = 0; k < K / 2; ++k) {
                        const V xnk = REMAT ? xnv[k] : ldg_v(xn_p + k * TSV);
                        const V xck = REMAT ? xcv[k] : ldg_v(xc_p + k * TSV);
                        const V ov = vfma(e_scale, packv(mine + k * VW), vfma(w, xnk, vmul(e_bee, xck)));
                        nrm += vnorm2(ov);
                        stcs_v(o2 + k * TSV, ov);
                    }
                } else {
#pragma unroll
                    for (int k = 0; k < K / 2; ++k) stcs_v(o2 + k * TSV, packv(mine + k * VW));
                }
            }
            if constexpr (EPI != 0) {
                if (++sl == Ls0) {
                    // |out|^2 of this (system, tile): fixed-tree sum over the consumer threads into partials[rhs][tile] --
                    // independent of which CTA took the tile, so the reduction is bit-reproducible under the dynamic queue
                    if (a.epi.partials != nullptr) {
#pragma unroll
                        for (int o2 = 16; o2 > 0; o2 >>= 1) nrm += __shfl_xor_sync(0xffffffffu, nrm, o2);
                        if (lane == 0) wsum[cw] = nrm;
                        asm volatile("bar.sync 1, %0;" ::"n"(128 * TPS) : "memory");
                        if (ctid == 0) {
                            double t = 0.0;
#pragma unroll
                            for (int i = 0; i < NCW; ++i) t += wsum[i];
                            a.epi.partials[(size_t)(s / Ls0) * ntiles + tile] = t;
                        }
                        asm volatile("bar.sync 1, %0;" ::"n"(128 * TPS) : "memory");      // wsum is free again
                        nrm = 0.0;
                    }
                    sl = 0;
                }
            }
        }
        tile = tile_next;
        ++j;
    }
}

// ------------------------------------------------------------------------------------------ launch
template <typename R, int TPS, int NG, int NST, int MINB, int EPI>
static dwf_status launch_tma_t(dwf_ctx* c, const TmaArgs& a, const CUtensorMap* maps, int* grid_out) {
    constexpr int K = VT<R>::K;
    const size_t smem = (size_t)NST * NREG * K * 512;
    auto kern = dhop_tma_kernel<R, TPS, NG, NST, MINB, EPI>;
    static unsigned long long attr_done = 0;      // per device (dwf_internal.h)
    if (attr_needed(attr_done, c->device))
        DWF_CUDA_CHECK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    TmaState* s = (TmaState*)c->tma;
    int grid = s->num_sms * MINB;
    if (grid > c->g.ntiles) grid = c->g.ntiles;
    if (grid_out) *grid_out = grid;
    kern<<<grid, 128 + 128 * TPS, smem, c->stream>>>(a, maps[0], maps[1], maps[2]);
    c->launches++;
    DWF_CUDA_CHECK(c, cudaGetLastError());
    return DWF_OK;
}

static dwf_status fill_args(dwf_ctx* c, TmaArgs& a, void* out, const void* in, int out_parity, int dagger, int prec,
                            const CUtensorMap** maps) {
    TmaState* s = (TmaState*)c->tma;
    dwf_status st = get_maps(c, in, prec, maps);
    if (st != DWF_OK) return st;
    memset(&a, 0, sizeof(a));
    a.g = geom_prec(c, prec, c->nrhs_cur); a.in = in; a.out = out;
    a.W = (prec == DWF_F64) ? c->W64[out_parity] : c->W32[out_parity];
    a.off = s->off + (size_t)(prec == DWF_F64 ? 0 : 2 * 8 * TSV) + (size_t)out_parity * 8 * TSV;
    a.gsrc = s->gsrc + (size_t)out_parity * 4 * 32;
    a.gdst = s->gdst + (size_t)out_parity * 4 * 32;
    a.xsrc = s->xsrc + (size_t)out_parity * 2 * 32;
    a.xdst = s->xdst + (size_t)out_parity * 2 * 32;
    a.order = s->order;
    a.counters = s->counters;
    a.mode = c->dhop_dynamic;
    a.dagger = dagger;
    a.epi.mode = EPI_NONE;
    return DWF_OK;
}

dwf_status launch_dhop_tma(dwf_ctx* c, void* out, const void* in, int out_parity, int dagger, int prec, bool* handled) {
    *handled = false;
    if (!c->tma) return DWF_OK;
    const CUtensorMap* maps = nullptr;
    TmaArgs a;
    dwf_status st = fill_args(c, a, out, in, out_parity, dagger, prec, &maps);
    if (st != DWF_OK) return st;
    *handled = true;
    if (prec == DWF_F64)
        return c->compress12 ? launch_tma_t<double, 2, 12, 3, 1, 0>(c, a, maps, nullptr)
                             : launch_tma_t<double, 2, 18, 3, 1, 0>(c, a, maps, nullptr);
    return c->compress12 ? launch_tma_t<float, 1, 12, 3, 2, 0>(c, a, maps, nullptr)
                         : launch_tma_t<float, 1, 18, 3, 2, 0>(c, a, maps, nullptr);
}

// the fused kernel exists for 4^4 tiles with 2-row links (any Ls)
bool dhop_fused_available(const dwf_ctx* c) { return c->tma != nullptr && c->fuse && c->compress12; }

// out = Mee xin + scale Dhop in (non-daggered), norm_slot >= 0: |out|^2 -> scalars[norm_slot]
dwf_status launch_dhop_fused(dwf_ctx* c, void* out, const void* in, int out_parity, int prec, const void* xin, double scale,
                             int norm_slot) {
    if (!dhop_fused_available(c)) { c->err = "fused Dhop kernel not available for this geometry"; return DWF_ESTATE; }
    const CUtensorMap* maps = nullptr;
    TmaArgs a;
    dwf_status st = fill_args(c, a, out, in, out_parity, 0, prec, &maps);
    if (st != DWF_OK) return st;
    const double bee = 1.0 + c->b5 * (4.0 - c->M5), cee = 1.0 - c->c5 * (4.0 - c->M5);
    EpiArgs& e = a.epi;
    e.mode = EPI_FINAL;
    e.xin = xin;
    e.bee = bee; e.mcee = -cee; e.mf = c->mf; e.scale = scale;
    e.Ls0 = c->g.Ls;
    int grid = 0;
    if (norm_slot >= 0) {
        st = ensure_partials(c, c->g.ntiles);              // one partial per tile
        if (st != DWF_OK) return st;
        e.partials = c->partials;
    }
    st = dhop_time_begin(c);
    if (st != DWF_OK) return st;
    st = (prec == DWF_F64) ? launch_tma_t<double, 2, 12, 3, 1, 1>(c, a, maps, &grid)
                           : launch_tma_t<float, 1, 12, 3, 2, 1>(c, a, maps, &grid);
    if (st != DWF_OK) return st;
    // algorithmic bytes: the input field, xin, the links, one field written
    const double B = (prec == DWF_F64) ? 8.0 : 4.0;
    st = dhop_time_end(c, 3.0 * (double)half_bytes(c->g, prec) * c->nrhs_cur + (double)c->g.Vh * 8 * 12 * B);
    if (st != DWF_OK) return st;
    if (norm_slot >= 0) return launch_reduce(c, c->g.ntiles, norm_slot, 0);
    return DWF_OK;
}

}  // namespace dwf
