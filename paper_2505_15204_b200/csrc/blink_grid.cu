// blink_grid: steps a0-a3.  One CTA per (timestep, channel): computes the nearest uv cell of every
// baseline (bit-exact twin of the oracle's fp32 recipe, R2), bins the samples and their
// Hermitian conjugates by ROW-BAND TILE of the grid (counting sort in shared memory), then for each
// band accumulates the tile in shared memory and stores it ONCE, zeros included -- no memset, no
// global atomics.  Only when a (t,c)'s binned list does not fit in shared memory are the baselines
// processed in chunks, and chunks after the first are added to the grid with global atomics (spill).
// PAPER.md L190-192 (gridding, no kernel, natural weighting); uniform weighting is reading R9.
#include "blink_common.cuh"

namespace blink {

constexpr int kGridThreads = 512;
constexpr int kTileCellsMax = 8192;               // 64 KB of complex64 per band tile

struct GridArgs {
    const float2 *vis; const float *uvw_m;
    int T, C, P, B, n, weighting;
    int tc0, c_base, out_tc0;                     // first flattened (t,c) of this launch; channel of s[0]; tc of grid[0]
    float2 *grid; float *wsum; int32_t *cell_idx; uint32_t *counts;     // wsum/cell_idx by absolute tc, grid/counts by tc - out_tc0
    int chunk_b, n_chunks, tile_cells, n_bands;
    int half_only;                                // the consumer only reads rows v >= 0 (Hermitian transform): skip the bands below
    int *row_extent;                              // OPTIONAL [tc - out_tc0]: rows v = 0 .. row_extent-1 are the only ones the consumer has to read;
                                                  // with half_only the (all-zero) bands above the last occupied one are not even stored
};

__global__ void __launch_bounds__(kGridThreads)
grid_tiles_kernel(const GridArgs a, const __grid_constant__ ScaleBlock sc)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2 *tile = reinterpret_cast<float2 *>(smem_raw);
    uint32_t *cnt = reinterpret_cast<uint32_t *>(tile + a.tile_cells);
    uint32_t *off = cnt + a.tile_cells;                        // [n_bands + 1]
    uint32_t *cur = off + a.n_bands + 1;                       // [n_bands]
    uint32_t *items = cur + a.n_bands;                         // [2 * chunk_b]
    __shared__ uint32_t red[kGridThreads / 32];
    __shared__ int s_last;                                     // last band that holds a sample (-1: none)

    const int tc = a.tc0 + blockIdx.x;
    const int t = tc / a.C, c = tc - t * a.C;
    const float s = sc.s[c - a.c_base];
    const int n = a.n, h = a.n / 2, B = a.B;
    const int tile_shift = 31 - __clz(a.tile_cells);
    const float *uvw = a.uvw_m + (size_t)t * B * 3;
    const size_t n2 = (size_t)n * n;
    const bool uniform = a.weighting == BLINK_W_UNIFORM;
    const bool multi = a.n_chunks > 1;
    const int otc = tc - a.out_tc0;
    uint32_t *gcounts = a.counts ? a.counts + (size_t)otc * n2 : nullptr;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    uint32_t my_in = 0, my_occ = 0;

    for (int ch = 0; ch < a.n_chunks; ++ch) {
        const int b0 = ch * a.chunk_b;
        const int b1 = min(B, b0 + a.chunk_b);
        // ---- phase 1: cell index of every baseline of the chunk, band histogram --------------------
        for (int i = threadIdx.x; i <= a.n_bands; i += kGridThreads) off[i] = 0;
        if (threadIdx.x == 0) s_last = -1;
        __syncthreads();
        for (int b = b0 + threadIdx.x; b < b1; b += kGridThreads) {
            const int cell = cell_of(uvw[3 * b], uvw[3 * b + 1], s, n, h);
            if (a.cell_idx) a.cell_idx[(size_t)tc * B + b] = cell;
            if (cell >= 0) {
                ++my_in;
                atomicAdd(&off[cell >> tile_shift], 1u);
                atomicAdd(&off[mirror_of(cell, n) >> tile_shift], 1u);
            }
        }
        __syncthreads();
        if (warp == 0) {                                       // exclusive scan of the band histogram
            uint32_t carry = 0;
            for (int base = 0; base < a.n_bands; base += 32) {
                const uint32_t v = (base + lane < a.n_bands) ? off[base + lane] : 0u;
                uint32_t inc = v;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) {
                    const uint32_t y = __shfl_up_sync(0xffffffffu, inc, d);
                    if (lane >= d) inc += y;
                }
                if (base + lane < a.n_bands) { off[base + lane] = carry + inc - v; cur[base + lane] = carry + inc - v; }
                carry += __shfl_sync(0xffffffffu, inc, 31);
            }
            if (lane == 0) off[a.n_bands] = carry;
        }
        __syncthreads();
        if (a.row_extent) {                                    // the occupied bands are mirror-symmetric: the last one bounds the rows v >= 0 in use
            int mine = -1;
            for (int i = threadIdx.x; i < a.n_bands; i += kGridThreads)
                if (off[i + 1] > off[i]) mine = i;             // increasing i per thread
            if (mine >= 0) atomicMax(&s_last, mine);
        }
        // ---- phase 2: counting-sort the samples (and conjugates) by band ---------------------------
        for (int b = b0 + threadIdx.x; b < b1; b += kGridThreads) {
            const int cell = cell_of(uvw[3 * b], uvw[3 * b + 1], s, n, h);
            if (cell >= 0) {
                const int mir = mirror_of(cell, n);
                const uint32_t bl = (uint32_t)(b - b0) << 14;
                uint32_t pos = atomicAdd(&cur[cell >> tile_shift], 1u);
                items[pos] = bl | (uint32_t)(cell & (a.tile_cells - 1));
                pos = atomicAdd(&cur[mir >> tile_shift], 1u);
                items[pos] = bl | (1u << 13) | (uint32_t)(mir & (a.tile_cells - 1));
            }
        }
        __syncthreads();
        // ---- phase 3: per band, per polarisation: accumulate in shared memory, store once ---------
        for (int band = 0; band < a.n_bands; ++band) {
            const uint32_t k0 = off[band], k1 = off[band + 1];
            if (multi && ch > 0 && k0 == k1) continue;         // nothing to spill for this band (uniform branch)
            if (a.half_only && (size_t)(band + 1) * a.tile_cells <= (size_t)h * n) continue;   // rows v < 0 only: never read
            // empty rows above the data are never read either; the band after the last occupied one is still stored because
            // the last row in use may straddle the band boundary (bands are 8192 cells, not whole rows)
            if (a.half_only && a.row_extent && band > s_last + 1) continue;
            for (int p = 0; p < a.P; ++p) {
                for (int i = threadIdx.x; i < a.tile_cells; i += kGridThreads) {
                    tile[i] = make_float2(0.f, 0.f);
                    if (p == 0) cnt[i] = 0u;
                }
                __syncthreads();
                const float2 *vrow = a.vis + ((size_t)tc * a.P + p) * B + b0;
                for (uint32_t k = k0 + threadIdx.x; k < k1; k += kGridThreads) {
                    const uint32_t it = items[k];
                    const int cl = it & 8191u;
                    float2 v = __ldg(vrow + (it >> 14));
                    if (it & (1u << 13)) v.y = -v.y;           // Hermitian conjugate sample
                    cell_add_exch(&tile[cl], v);              // native 64-bit exchanges instead of two fp32 CAS loops (blink_common.cuh)
                    if (p == 0) atomicAdd(&cnt[cl], 1u);
                }
                __syncthreads();
                float2 *gdst = a.grid + ((size_t)otc * a.P + p) * n2 + (size_t)band * a.tile_cells;
                // cells of this band that exist (n2 is a multiple of 4, so pairs / quads never straddle the end)
                const int tile_n = (int)min((size_t)a.tile_cells, n2 - (size_t)band * a.tile_cells);
                if (!multi) {
                    for (int i = threadIdx.x * 2; i < tile_n; i += kGridThreads * 2) {
                        float2 v0 = tile[i], v1 = tile[i + 1];
                        const uint32_t c0 = cnt[i], c1 = cnt[i + 1];
                        if (uniform) {
                            if (c0) { v0.x /= (float)c0; v0.y /= (float)c0; }
                            if (c1) { v1.x /= (float)c1; v1.y /= (float)c1; }
                        }
                        if (p == 0) {
                            if (!a.half_only) {
                                my_occ += (c0 != 0) + (c1 != 0);
                            } else {                            // occupied cells of the full plane from the rows v >= 0:
                                const size_t gi = (size_t)band * a.tile_cells + i;      // row v = 0 mirrors onto itself, rows v > 0 count twice
                                if (gi >= (size_t)h * n) my_occ += ((c0 != 0) + (c1 != 0)) * (gi < (size_t)(h + 1) * n ? 1 : 2);
                            }
                        }
                        __stcs(reinterpret_cast<float4 *>(gdst + i), make_float4(v0.x, v0.y, v1.x, v1.y));
                    }
                } else if (ch == 0) {
                    for (int i = threadIdx.x * 2; i < tile_n; i += kGridThreads * 2)
                        *reinterpret_cast<float4 *>(gdst + i) = make_float4(tile[i].x, tile[i].y, tile[i + 1].x, tile[i + 1].y);
                } else {                                        // spill: add the touched cells with global atomics
                    for (int i = threadIdx.x; i < tile_n; i += kGridThreads)
                        if (cnt[i]) { atomicAdd(&gdst[i].x, tile[i].x); atomicAdd(&gdst[i].y, tile[i].y); }
                }
                if (p == 0 && gcounts) {
                    uint32_t *cdst = gcounts + (size_t)band * a.tile_cells;
                    if (!multi || ch == 0) {
                        for (int i = threadIdx.x * 4; i < tile_n; i += kGridThreads * 4)
                            *reinterpret_cast<uint4 *>(cdst + i) = *reinterpret_cast<const uint4 *>(cnt + i);
                    } else {
                        for (int i = threadIdx.x; i < tile_n; i += kGridThreads)
                            if (cnt[i]) atomicAdd(&cdst[i], cnt[i]);
                    }
                }
                __syncthreads();
            }
        }
        if (multi) { __threadfence(); __syncthreads(); }       // this CTA's stores/atomics ordered before the next chunk
    }
    // ---- multi-chunk uniform weighting: divide by the final counts (kept in global memory) ---------
    if (multi && (uniform)) {
        for (size_t i = threadIdx.x; i < n2; i += kGridThreads) {
            const uint32_t cc = gcounts[i];
            if (cc) {
                ++my_occ;
                for (int p = 0; p < a.P; ++p) {
                    float2 *g = a.grid + ((size_t)otc * a.P + p) * n2 + i;
                    float2 v = *g;
                    v.x /= (float)cc; v.y /= (float)cc;
                    *g = v;
                }
            }
        }
    }
    if (a.row_extent && threadIdx.x == 0) {
        // rows v >= 0 (centred rows h .. h + extent - 1) that lie in bands 0 .. s_last; everything above is zero / not stored
        int ext = h;
        if (a.half_only) {
            const long long last_cell = (long long)(s_last + 1) * a.tile_cells - 1;            // -1 when there is no sample at all
            const long long r = last_cell < 0 ? -1 : last_cell / n;
            ext = (int)(r - h + 1);
            ext = ext < 0 ? 0 : (ext > h ? h : ext);
        }
        a.row_extent[otc] = ext;
    }
    // ---- weight sum ----------------------------------------------------------------------------
    uint32_t val = uniform ? my_occ : my_in;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) val += __shfl_xor_sync(0xffffffffu, val, d);
    if (lane == 0) red[warp] = val;
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t tot = 0;
        for (int w = 0; w < kGridThreads / 32; ++w) tot += red[w];
        a.wsum[tc] = uniform ? (float)tot : (float)(2u * tot);
    }
}

// band tile: a power of two number of cells (the band of a cell is a shift), at most 8192
static int grid_tile_cells(size_t n2)
{
    int t = kTileCellsMax;
    while ((size_t)t > n2) t >>= 1;
    return t;
}
static size_t grid_smem_bytes(int tile_cells, int n_bands, int chunk_b)
{
    return (size_t)tile_cells * 12 + (size_t)(2 * n_bands + 1) * 4 + (size_t)chunk_b * 8 + 16;
}

// baselines per chunk that fit next to the tile in 227 KB of shared memory
static int grid_chunk_capacity(int n_pix)
{
    const size_t n2 = (size_t)n_pix * n_pix;
    const int tile_cells = grid_tile_cells(n2);
    const int n_bands = (int)((n2 + tile_cells - 1) / tile_cells);
    const size_t fixed = grid_smem_bytes(tile_cells, n_bands, 0);
    const size_t avail = 227 * 1024 - 1024 - fixed;
    size_t cap = avail / 8;
    if (cap > (size_t)kMaxBaselines) cap = kMaxBaselines;
    return (int)cap;
}

bool grid_needs_global_counts(int B, int n_pix, int weighting)
{
    int chunk = option(BLINK_OPT_GRID_CHUNK_B);
    if (chunk <= 0) chunk = grid_chunk_capacity(n_pix);
    return weighting == BLINK_W_UNIFORM && B > chunk;
}

// Tiny batches (a single image, a handful of them): one CTA per (t,c) leaves the other SMs idle -- 52 of the 67 us of BASELINE
// config 1 (one 256 x 256 image) were this gridder on ONE SM.  Natural weighting only: the grids are zeroed by a memset and every
// (baseline, (t,c)) thread adds its sample and the conjugate with `red.global.add.v2.f32`; the in-range count of a (t,c) is
// collected in its wsum slot as an integer (warp ballot + one atomic per warp) and turned into W = 2 count by a finishing kernel.
__global__ void __launch_bounds__(256)
grid_scatter_small_kernel(const GridArgs a, const __grid_constant__ ScaleBlock sc)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    const int tc = a.tc0 + blockIdx.y;
    const int t = tc / a.C, c = tc - t * a.C;
    const int n = a.n;
    const size_t n2 = (size_t)n * n;
    bool in = false;
    if (b < a.B) {
        const float *uvw = a.uvw_m + ((size_t)t * a.B + b) * 3;
        const int cell = cell_of(uvw[0], uvw[1], sc.s[c - a.c_base], n, n / 2);
        if (a.cell_idx) a.cell_idx[(size_t)tc * a.B + b] = cell;
        if (cell >= 0) {
            in = true;
            const int mir = mirror_of(cell, n);
            const int otc = tc - a.out_tc0;
            for (int p = 0; p < a.P; ++p) {
                const float2 v = __ldg(a.vis + ((size_t)tc * a.P + p) * a.B + b);
                float2 *g = a.grid + ((size_t)otc * a.P + p) * n2;
                atomicAdd(&g[cell], v);
                atomicAdd(&g[mir], make_float2(v.x, -v.y));
            }
        }
    }
    const unsigned m = __ballot_sync(0xffffffffu, in);
    if ((threadIdx.x & 31) == 0 && m) atomicAdd(reinterpret_cast<unsigned *>(a.wsum) + tc, (unsigned)__popc(m));
}
__global__ void grid_scatter_finish_kernel(float *wsum, int tc0, int ntc)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ntc) wsum[tc0 + i] = (float)(2u * reinterpret_cast<const unsigned *>(wsum)[tc0 + i]);
}

int grid_range(const float2 *vis, const float *uvw_m, const double *freqs_hz, double pixscale_rad, int T, int C, int P,
               int B, int n_pix, int weighting, int tc0, int ntc, int out_tc0, float2 *grid, float *wsum,
               int32_t *cell_idx, uint32_t *counts, cudaStream_t st, bool half_only, int *row_extent)
{
    (void)T;
    if (ntc <= 0) return BLINK_OK;
    const size_t n2 = (size_t)n_pix * n_pix;
    GridArgs a;
    a.vis = vis; a.uvw_m = uvw_m; a.T = T; a.C = C; a.P = P; a.B = B; a.n = n_pix; a.weighting = weighting;
    a.out_tc0 = out_tc0; a.grid = grid; a.wsum = wsum; a.cell_idx = cell_idx; a.counts = counts;
    a.tile_cells = grid_tile_cells(n2);
    a.n_bands = (int)((n2 + a.tile_cells - 1) / a.tile_cells);          // the last band may be partial (sides that are not a power of two)
    int chunk = option(BLINK_OPT_GRID_CHUNK_B);
    const int cap = grid_chunk_capacity(n_pix);
    if (chunk <= 0 || chunk > cap) chunk = cap;
    if (chunk > B) chunk = B > 0 ? B : 1;
    a.chunk_b = chunk;
    a.n_chunks = B > 0 ? (B + chunk - 1) / chunk : 1;
    if (a.n_chunks > 1 && weighting == BLINK_W_UNIFORM && counts == nullptr) return BLINK_ERR_WORKSPACE;
    a.half_only = (half_only && a.n_chunks == 1 && counts == nullptr) ? 1 : 0;
    a.row_extent = row_extent;
    // tiny batches, natural weighting, nothing but the plain outputs asked for: scatter with global atomics over all SMs
    const bool small = weighting == BLINK_W_NATURAL && counts == nullptr && !half_only && row_extent == nullptr &&
                       ntc <= 128 && C <= 1024 && option(BLINK_OPT_GRID_CHUNK_B) == 0;
    if (small) {
        BLINK_CUDA_TRY(cudaMemsetAsync(grid + (size_t)(tc0 - out_tc0) * P * n2, 0, (size_t)ntc * P * n2 * sizeof(float2), st));
        BLINK_CUDA_TRY(cudaMemsetAsync(wsum + tc0, 0, (size_t)ntc * sizeof(float), st));
        ScaleBlock sc;
        for (int k = 0; k < 1024; ++k) sc.s[k] = k < C ? scale_for(freqs_hz[k], n_pix, pixscale_rad) : 0.f;
        a.tc0 = tc0; a.c_base = 0;
        grid_scatter_small_kernel<<<dim3((unsigned)((B + 255) / 256), (unsigned)ntc), 256, 0, st>>>(a, sc);
        BLINK_LAUNCH_CHECK("grid_scatter_small_kernel");
        grid_scatter_finish_kernel<<<(ntc + 63) / 64, 64, 0, st>>>(wsum, tc0, ntc);
        BLINK_LAUNCH_CHECK("grid_scatter_finish_kernel");
        return BLINK_OK;
    }
    const size_t smem = grid_smem_bytes(a.tile_cells, a.n_bands, a.chunk_b);
    BLINK_CUDA_TRY(cudaFuncSetAttribute(grid_tiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    // sub-ranges that stay inside one timestep's block of <= 1024 channels (scales travel as a kernel parameter)
    int tc = tc0;
    const int tc_end = tc0 + ntc;
    while (tc < tc_end) {
        const int t = tc / C, c = tc - t * C;
        const int c_base = (c / 1024) * 1024;
        const int c_lim = c_base + 1024 < C ? c_base + 1024 : C;
        int end = t * C + c_lim;
        if (C <= 1024) end = tc_end;                          // one block covers every timestep
        if (end > tc_end) end = tc_end;
        ScaleBlock sc;
        for (int k = 0; k < 1024; ++k) sc.s[k] = (c_base + k < C) ? scale_for(freqs_hz[c_base + k], n_pix, pixscale_rad) : 0.f;
        a.tc0 = tc; a.c_base = c_base;
        grid_tiles_kernel<<<end - tc, kGridThreads, smem, st>>>(a, sc);
        BLINK_LAUNCH_CHECK("grid_tiles_kernel");
        tc = end;
    }
    return BLINK_OK;
}

}  // namespace blink

extern "C" int blink_grid(const blink_c64 *vis, const float *uvw_m, const double *freqs_hz, int T, int C, int P, int B,
                          int n_pix, double pixscale_rad, int weighting, blink_c64 *grid, float *wsum,
                          int32_t *cell_idx, uint32_t *counts, void *workspace, size_t workspace_bytes, void *stream)
{
    using namespace blink;
    if (!vis || !uvw_m || !freqs_hz || !grid || !wsum) return BLINK_ERR_INVALID_ARG;
    if (T < 1 || C < 1 || P < 1 || B < 1 || !(pixscale_rad > 0.0)) return BLINK_ERR_INVALID_ARG;
    if (weighting != BLINK_W_NATURAL && weighting != BLINK_W_UNIFORM) return BLINK_ERR_INVALID_ARG;
    if (!aligned16(vis) || !aligned16(grid) || (counts && !aligned16(counts))) return BLINK_ERR_INVALID_ARG;
    if (!size_supported(n_pix) || B > kMaxBaselines) return BLINK_ERR_UNSUPPORTED;
    if ((long long)T * C > 0x7fffffffLL / 2) return BLINK_ERR_UNSUPPORTED;
    int rc = ensure_device();
    if (rc != BLINK_OK) return rc;
    uint32_t *counts_eff = counts;
    if (!counts && grid_needs_global_counts(B, n_pix, weighting)) {
        const size_t need = (size_t)T * C * n_pix * n_pix * sizeof(uint32_t);
        if (!workspace || workspace_bytes < need || !aligned16(workspace)) return BLINK_ERR_WORKSPACE;
        counts_eff = static_cast<uint32_t *>(workspace);
    }
    return grid_range(reinterpret_cast<const float2 *>(vis), uvw_m, freqs_hz, pixscale_rad, T, C, P, B, n_pix,
                      weighting, 0, T * C, 0, reinterpret_cast<float2 *>(grid), wsum, cell_idx, counts_eff,
                      static_cast<cudaStream_t>(stream));
}
