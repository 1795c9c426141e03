// cfs_bin.cuh -- tile-binned splat stage (sm_100a): the way past the L2 atomic rate.
//
// A direct splat costs one L2 reduction (row 7), and the L2 executes ~190 G of them per second
// whatever their width (measured, cfs_microbench) -- 3x below what the sampler can generate.
// Shared-memory privatisation removes that bound, but no BASELINE image fits one CTA's shared
// memory (SURVEY 7 "hard parts" 1).  So the image is cut into tiles that do fit -- INTERLEAVED ones: with 2^t tiles,
// pixel p belongs to tile p & (2^t - 1) as its pixel p >> t, so every tile samples the whole image and all tiles draw
// splats at the same rate -- and the splats are partitioned by tile on their way through HBM:
//
//   pass 1 (render_kernel<..., SPLAT_BIN>): each splat becomes ONE 16-bit record
//     (colour index * pixels per tile + pixel-in-tile), appended with one shared-memory atomic to the CTA's
//     staging row of its tile; every ~100 iterations the rows are drained by the bulk-copy engine (cp.async.bulk
//     shared -> global) into 2 KiB pool blocks owned by (CTA, tile), so no global atomic is paid per splat -- one
//     per 1024 records.
//   pass 2 (bin_accumulate_kernel): one CTA per (tile, part) walks the tile's block list with
//     coalesced 128-bit loads and counts records with shared-memory atomics (the record IS the
//     counter index), then merges its private tile into the image with one red.global per
//     touched pixel: "per-CTA shared-memory privatised histograms merged with red.global"
//     (BASELINE north_star), made to work for images of any size.
//
// Nothing here can lose a splat: a staging row, the block pool or a tile list running out sends
// the affected records down the direct path (one L2 reduction each).
#pragma once
#include "cfs_device.cuh"

namespace cfs {

__device__ __forceinline__ void bin_red_add_v4_f32(float *addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};"
                 :: "l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}

__device__ __forceinline__ void bin_red_add_u32(uint32_t *addr, uint32_t v)
{
    asm volatile("red.global.add.u32 [%0], %1;" :: "l"(addr), "r"(v) : "memory");
}

// shared-memory layout of pass 1 (dynamic): u32 cnt[n_tiles + kBinDummy] | pad to 16 B | u16 buf[n_tiles][cap].  The
// fill counters are contiguous on purpose: 32 lanes taking slots in 32 random tiles spread over all 32 banks (a
// counter at the head of each row puts them all on 8 banks: rows are a multiple of 128 bytes apart plus the head;
// measured slower, 3.19 against 2.96 ms on configs[1]).  cnt[n_tiles + lane] is lane's DUMMY counter, pre-set to the
// row capacity: a dropped splat takes its slot there and so finds "no room" -- the append stays straight-line code
// (a predicated atom.shared compiles to a branch around it: three more instructions per splat, measured) and the
// dropped splats of different lanes never meet on one address.
__device__ __forceinline__ uint32_t bin_buf_offset(uint32_t n_tiles) { return (n_tiles + kBinDummy + 3u) & ~3u; }

// one record down the direct path (staging row full, or no pool block for the tile)
__device__ __forceinline__ void bin_direct(const RenderParams &prm, const SharedTables &s, uint32_t tile, uint32_t rec)
{
    const uint32_t pix = ((rec % prm.bin.tile_pixels) << prm.bin.tshift) | tile;   // rare path: a real division is fine
    if (prm.color_rule == 0) {
        bin_red_add_u32(reinterpret_cast<uint32_t *>(prm.image) + pix, 1u);
    } else {
        const float4 c = s.palette[rec / prm.bin.tile_pixels];
        bin_red_add_v4_f32(reinterpret_cast<float *>(prm.image) + 4 * (size_t)pix, c.x, c.y, c.z, c.w);   // c.w = 1 (load_tables)
    }
}

// values of the append fast path, derived once per thread (32-bit shared-window addresses, so
// an access is one ATOMS / STS without generic-address arithmetic)
struct BinRegs {
    uint32_t cnt_addr, buf_addr;   // shared addresses of cnt[] and buf[][]
    uint32_t row_bytes, cap;       // bytes per row, records per row
    uint32_t dummy;                // index of this lane's dummy counter (n_tiles + lane)
    uint32_t tmask, tshift;        // tile of pixel p = p & tmask, its pixel in the tile p >> tshift (interleaved tiles)
    uint32_t ktp;                  // colour index stride of a record: tp for RGBA, 0 for HIST (the colour is ignored)
    float sx, ox, sy, oy;          // pixel map (DESIGN R8)
    float xmin, xmax, ymin, ymax;  // closed bounds (DESIGN R8)
    int W, Wm1, Hm1;
};

__device__ __forceinline__ BinRegs bin_regs_init(const RenderParams &prm, uint32_t *sm)
{
    BinRegs r;
    r.cnt_addr = (uint32_t)__cvta_generic_to_shared(sm);
    r.buf_addr = r.cnt_addr + 4u * bin_buf_offset(prm.bin.n_tiles);
    r.cap = prm.bin.cap; r.row_bytes = 2u * prm.bin.cap + kBinRowPad;
    r.dummy = prm.bin.n_tiles;      // + lane, added by each thread after the broadcast
    r.tmask = prm.bin.tmask; r.tshift = prm.bin.tshift;
    r.ktp = (prm.color_rule == 0) ? 0u : prm.bin.tile_pixels;
    r.sx = prm.sx; r.ox = prm.ox; r.sy = prm.sy; r.oy = prm.oy;
    r.xmin = prm.xmin; r.xmax = prm.xmax; r.ymin = prm.ymin; r.ymax = prm.ymax;
    r.W = prm.W; r.Wm1 = prm.W - 1; r.Hm1 = prm.H - 1;
    return r;
}

// bounds rule of cfs_device.cuh in_bounds(), operands from registers.  SYM: the bounds are symmetric about 0
// (host-checked), so the closed test is two compares on |x|, |y| -- the same truth value for every float, NaN included.
template <bool SYM>
__device__ __forceinline__ bool bin_in_bounds(const BinRegs &br, float x, float y)
{
    if (SYM) return (fabsf(x) <= br.xmax) && (fabsf(y) <= br.ymax);
    return (x >= br.xmin) && (x <= br.xmax) && (y >= br.ymin) && (y <= br.ymax);
}

// pixel rule of cfs_device.cuh pixel_of(), operands from registers
// (the unsigned conversion saturates negative values to 0: the lower clamp costs nothing)
// UNCLAMPED: the host has proved every splat inside the bounds with a margin (OPT_NO_DROP): the upper clamp cannot
// bind; a thread without a point (NaN) converts to pixel 0 and stores nothing
template <bool UNCLAMPED = false>
__device__ __forceinline__ int bin_pixel_of(const BinRegs &br, float x, float y)
{
    uint32_t px = __float2uint_rd(__fmaf_rn(x, br.sx, br.ox));
    uint32_t py = __float2uint_rd(__fmaf_rn(y, br.sy, br.oy));
    CFS_CHECK(!UNCLAMPED || (px <= (uint32_t)br.Wm1 && py <= (uint32_t)br.Hm1));
    if (!UNCLAMPED) { px = min(px, (uint32_t)br.Wm1); py = min(py, (uint32_t)br.Hm1); }
    return (int)(py * (uint32_t)br.W + px);
}

__device__ __forceinline__ void bin_record_of(const BinRegs &br, int pix, int k, uint32_t &tile, uint32_t &rec)
{
    tile = (uint32_t)pix & br.tmask;
    rec = ((uint32_t)pix >> br.tshift) + (uint32_t)k * br.ktp;
}

// row 7, binned: one shared-memory atomic + one shared store per splat (interpreter path: branches are fine here)
__device__ __forceinline__ void bin_append(const RenderParams &prm, const SharedTables &s, const BinRegs &br, int pix, int k)
{
    uint32_t tile, rec;
    bin_record_of(br, pix, k, tile, rec);
    CFS_CHECK(tile < prm.bin.n_tiles && rec < prm.bin.tile_pixels * prm.bin.nk);
    const uint32_t row = br.buf_addr + tile * br.row_bytes;
    uint32_t slot;
    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(slot) : "r"(br.cnt_addr + 4u * tile) : "memory");
    if (slot < br.cap) asm volatile("st.shared.u16 [%0], %1;" :: "r"(row + 2u * slot), "h"((uint16_t)rec) : "memory");
    else bin_direct(prm, s, tile, rec);
}

// The same as straight-line code, in two halves (the caller issues the atomics of a whole Philox block before the
// first store, so their latencies overlap).  A dropped splat takes its slot from the lane's dummy counter, which always
// reads "full", so the store is predicated on the slot alone.  bin_store_record returns true when the record was stored;
// false means "row full" -- a live record then has to go down the direct path (rare; the caller does that afterwards
// and tells live from dropped by `ok`).
__device__ __forceinline__ uint32_t bin_take_slot(const BinRegs &br, bool ok, uint32_t tile, uint32_t rec)
{
    const uint32_t t_eff = ok ? tile : br.dummy;
    CFS_CHECK(tile <= br.dummy - (threadIdx.x & 31u) - 1u && rec <= 49152u);
    uint32_t slot;
    asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(slot) : "r"(br.cnt_addr + 4u * t_eff) : "memory");
    return slot;
}
__device__ __forceinline__ bool bin_store_record(const BinRegs &br, uint32_t tile, uint32_t rec, uint32_t slot)
{
    const bool fits = slot < br.cap;
    if (fits) asm volatile("st.shared.u16 [%0], %1;" :: "r"(br.buf_addr + tile * br.row_bytes + 2u * slot), "h"((uint16_t)rec) : "memory");
    return fits;
}
// Per-lane bin state of pass 1, kept in REGISTERS: lane l of warp w owns tile l * warps + w (so
// n_tiles <= 32 * warps per CTA, and the rows to flush are spread over all warps of the CTA).  `next` is a pool block taken ahead of time: the global atomic
// that hands it out is issued when the previous block is opened and its result is not needed
// until that block is full, so its latency never sits between the two barriers of a flush.
struct BinLane {
    uint32_t pos;    // next record position in the pool (block * 512 + fill); 0 = no block yet
    uint32_t next;   // prefetched block id
    uint32_t nblk;   // blocks this CTA has listed for the tile
};

__device__ __forceinline__ void bin_lane_init(const RenderParams &prm, BinLane &bl)
{
    bl.pos = 0u; bl.nblk = 0u;
    const uint32_t my_tile = (threadIdx.x & 31u) * (blockDim.x >> 5) + (threadIdx.x >> 5);
    bl.next = (my_tile < prm.bin.n_tiles) ? atomicAdd(&prm.bin.ctrl[0], 1u) + 1u : 0u;   // block 0 is never used
}

// The staging records are written through the generic proxy (st.shared) and read by the bulk-copy engine (async
// proxy): every WRITER orders its stores with this fence, then the threads synchronise, then one lane issues the copy
// (render_kernel fences before the barrier that precedes bin_drain).
__device__ __forceinline__ void bin_fence_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// Called by every thread of the CTA between two __syncthreads: the owning warp DRAINS every staging row that holds at
// least kBinDrainMin records (any record when `final`) into the (CTA, tile) pool block -- the WHOLE row, padded to a whole
// 128-bit vector with the DUMMY record (the counter behind the tile's last one: pass 2 counts it without a test), moved
// by the bulk-copy engine: one elected lane hands the row to cp.async.bulk (shared -> global, split where it crosses
// into the next 2 KiB block), so no lane loads or stores a record and nothing stays behind -- no remainder to move, all
// of a row's capacity serves the next interval.  The warp then waits until the engine has READ the rows (not for the
// writes to land; the final drain waits for those).  A tile whose pool or list ran out sends its records down the
// direct path.  (History: whole 256-record units through LDS.128 -> STG.128 by all 32 lanes, with the remainder carried,
// were 10.8 % of the instructions of pass 1; the same units through the bulk engine 12 % less time on configs[2].)
__device__ __forceinline__ void bin_drain(const RenderParams &prm, const SharedTables &s, const BinRegs &br, BinLane &bl, bool final)
{
    const BinParams &b = prm.bin;
    constexpr uint32_t nwarps = (uint32_t)kBinThreads / 32u;      // pass 1 is always launched with kBinThreads threads
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    if (warp >= b.n_tiles) return;                     // warp owns no tile (warp-uniform)
    const uint32_t my_tile = lane * nwarps + warp;
    const bool valid = my_tile < b.n_tiles;
    uint32_t mine = 0u;
    if (valid) asm volatile("ld.shared.u32 %0, [%1];" : "=r"(mine) : "r"(br.cnt_addr + 4u * my_tile));
    mine = min(mine, br.cap);                          // slots >= cap went direct
    unsigned todo = __ballot_sync(0xFFFFFFFFu, final ? mine > 0u : mine >= b.drain_min);
    if (todo != 0u) {
        const size_t list_base = ((size_t)my_tile * b.grid + blockIdx.x) * b.lcap;
        const uint32_t dummy = b.tile_pixels * b.nk;
        do {
            const int src = __ffs(todo) - 1;
            todo &= todo - 1;
            const uint32_t tile = (uint32_t)src * nwarps + warp;
            const uint32_t cnt = __shfl_sync(0xFFFFFFFFu, mine, src);
            const uint32_t cnt8 = (cnt + kBinGrain - 1u) & ~(kBinGrain - 1u);     // <= cap: cap is a multiple of 64
            const uint32_t row = br.buf_addr + tile * br.row_bytes;
            if (cnt + lane < cnt8)                                            // pad the last vector (at most 7 records)
                asm volatile("st.shared.u16 [%0], %1;" :: "r"(row + 2u * (cnt + lane)), "h"((uint16_t)dummy) : "memory");
            bin_fence_async();                                                // writers fence, then synchronise, then one lane issues
            __syncwarp();
            uint32_t left = cnt8, from = row;
            do {
                uint32_t pos = __shfl_sync(0xFFFFFFFFu, bl.pos, src);
                if ((pos & (kBinBlockRecords - 1u)) == 0u) {                  // block full (or none yet); kBinInvalid ends in ones
                    if ((int)lane == src) {    // open the prefetched block, list it, prefetch another
                        if (bl.next < b.nb && bl.nblk < b.lcap) {
                            b.list[list_base + bl.nblk] = bl.next;
                            bl.pos = bl.next * kBinBlockRecords;
                            ++bl.nblk;
                            bl.next = atomicAdd(&b.ctrl[0], 1u) + 1u;
                        } else {
                            bl.pos = kBinInvalid;              // pool or list exhausted: direct from now on
                        }
                    }
                    pos = __shfl_sync(0xFFFFFFFFu, bl.pos, src);
                }
                if (pos == kBinInvalid) {                                     // rare: the rest of the row goes down the direct path
                    const uint32_t first = cnt8 - left;
                    for (uint32_t i = first + lane; i < cnt; i += 32u) bin_direct(prm, s, tile, lds_u16(row + 2u * i));
                    if (lane == 0u && cnt > first) atomicAdd(&b.ctrl[1], cnt - first);
                    break;
                }
                const uint32_t seg = min(left, kBinBlockRecords - (pos & (kBinBlockRecords - 1u)));
                CFS_CHECK(pos >= kBinBlockRecords && pos + seg <= (b.nb + 1u) * kBinBlockRecords && (pos & (kBinGrain - 1u)) == 0u && (seg & (kBinGrain - 1u)) == 0u);
                CFS_CHECK(from + 2u * seg <= br.buf_addr + b.n_tiles * br.row_bytes);
                if (lane == 0u)
                    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                                 :: "l"(b.pool + pos), "r"(from), "r"(2u * seg) : "memory");
                if ((int)lane == src) bl.pos = pos + seg;
                from += 2u * seg;
                left -= seg;
            } while (left != 0u);
            if ((int)lane == src) mine = 0u;
        } while (todo != 0u);
        if (lane == 0u) {
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");     // the rows have been read: their memory is free again
        }
        __syncwarp();
    }
    if (final && lane == 0u) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");    // every record this warp handed over (now or in
                                                                                          // an earlier drain) has landed in the pool
    if (valid) asm volatile("st.shared.u32 [%0], %1;" :: "r"(br.cnt_addr + 4u * my_tile), "r"(mine) : "memory");
    if (final && valid) {
        // blocks listed for (tile, CTA) and the fill of the last one (a full block reads 1024)
        uint32_t fill = 0u;
        if (bl.nblk > 0u && bl.pos != kBinInvalid) {
            fill = bl.pos & (kBinBlockRecords - 1u);
            if (fill == 0u) fill = kBinBlockRecords;
        } else if (bl.nblk > 0u) {
            fill = kBinBlockRecords;                   // went invalid only after full blocks
        }
        b.tails[(size_t)my_tile * b.grid + blockIdx.x] = (bl.nblk << kBinTailShift) | fill;
    }
}

// ---------------------------------------------------------------------------------------------
// pass 2.  MODE 0: HIST_U32 (nk = 1).  MODE 1: RGBA_F32 + MAP_INDEX: counters per (colour index, pixel), laid
// out [k][pixel] -- the colour of a splat follows its position (the last map decides the region), so a tile is
// mostly ONE colour and a [pixel][k] layout would leave all records of a warp on 32 / nk banks (measured 5.2
// wavefronts per ATOMS in r01k); with [k][pixel] the bank is the pixel's.  The pixel's sum is
// sum_k n_k * palette[k] (any summation order is a correct result, DESIGN R8; exact for integer-valued palettes
// while every sum stays < 2^24).
//
// A record IS the index of its counter, and the pool holds whole 128-bit vectors of 8 records (pass 1 pads a
// drained row with the DUMMY record, the counter behind the tile's last one), so the count loop is three
// instructions per record: extract 16 bits, scale to a shared-window address, red.shared.add.
// Counter r lives at slot r ^ ((r >> 5) & 31): a permutation inside every aligned group of 32 counters that mixes
// bits 5..9 of the index into the bank.  The bank of a record was (pixel >> t) mod 32 -- on configs[1] a function of
// the coarse x position and y mod 4, and the swirled disc does not fill the x range evenly: 4.16 wavefronts per
// red.shared against 3.5 for uniformly random banks (and 3.6 on configs[2]).  Two more ALU instructions per record
// in a kernel that waits for the shared-memory pipe.
__device__ __forceinline__ uint32_t bin_slot(uint32_t r) { return r ^ ((r >> 5) & 31u); }
__device__ __forceinline__ void bin_count8(uint32_t acc_addr, const uint4 &v)
{
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        CFS_CHECK((w[i] & 0xFFFFu) <= 49152u && (w[i] >> 16) <= 49152u);
        asm volatile("red.shared.add.u32 [%0], 1;" :: "r"(acc_addr + (bin_slot(w[i] & 0xFFFFu) << 2)) : "memory");
        asm volatile("red.shared.add.u32 [%0], 1;" :: "r"(acc_addr + (bin_slot(w[i] >> 16) << 2)) : "memory");
    }
}

template <int MODE>
__global__ void __launch_bounds__(kBinAccThreads)
bin_accumulate_kernel(const __grid_constant__ RenderParams prm)
{
    extern __shared__ __align__(16) uint32_t acc[];     // tile_pixels * nk counters + the dummy one, rounded up to whole groups of 32 (bin_slot)
    const BinParams &b = prm.bin;
    const uint32_t tile = blockIdx.x / b.split, part = blockIdx.x % b.split;
    const uint32_t n_ctr = b.tile_pixels * b.nk;
    {
        uint4 *a4 = reinterpret_cast<uint4 *>(acc);
        for (uint32_t i = threadIdx.x; i < (n_ctr + 32u) / 32u * 8u; i += blockDim.x) a4[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    const uint32_t acc_addr = (uint32_t)__cvta_generic_to_shared(acc);

    // CTA `part` takes blocks j = part (mod split) of every pass-1 CTA's list for this tile; its
    // warps stripe over the pass-1 CTAs
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    for (uint32_t c = warp; c < b.grid; c += nwarps) {
        const uint32_t tail = b.tails[(size_t)tile * b.grid + c];
        const uint32_t n_blk = tail >> kBinTailShift, last_fill = tail & ((1u << kBinTailShift) - 1u);
        const uint32_t *list = b.list + ((size_t)tile * b.grid + c) * b.lcap;
        // two blocks (2 x 2 KiB, eight 128-bit loads per lane) in flight per warp; every block of a list is full except
        // the last, whose fill is a whole number of 128-bit vectors (bin_drain pads with the DUMMY record)
        for (uint32_t j = part; j < n_blk; j += 2u * b.split) {
            uint4 v[2][4];
            uint32_t nrec[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const uint32_t jj = j + (uint32_t)h * b.split;
                nrec[h] = 0u;
                if (jj < n_blk) {
                    nrec[h] = (jj + 1u == n_blk) ? last_fill : kBinBlockRecords;
                    const uint4 *src = reinterpret_cast<const uint4 *>(b.pool + (size_t)list[jj] * kBinBlockRecords);
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (kBinGrain * ((uint32_t)q * 32u + lane) < nrec[h]) v[h][q] = __ldcs(src + q * 32 + lane);
                }
            }
#pragma unroll
            for (int h = 0; h < 2; ++h) {
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (kBinGrain * ((uint32_t)q * 32u + lane) < nrec[h]) bin_count8(acc_addr, v[h][q]);
            }
        }
    }
    __syncthreads();

    // merge the private tile (red.global, touched pixels only)
    const uint32_t n_pix_tile = b.tile_pixels;
    const uint32_t n_pix = (uint32_t)prm.W * (uint32_t)prm.H, tshift = b.tshift;    // pixel i of the tile is image pixel (i << tshift) | tile
    if (MODE == 0) {
        uint32_t *hist = reinterpret_cast<uint32_t *>(prm.image);
        for (uint32_t i = threadIdx.x; i < n_pix_tile; i += blockDim.x) {
            const uint32_t c = acc[bin_slot(i)];
            const uint32_t pix = (i << tshift) | tile;
            if (c && pix < n_pix) bin_red_add_u32(hist + pix, c);
        }
    } else {
        float *img = reinterpret_cast<float *>(prm.image);
        const uint32_t nk = b.nk;
        for (uint32_t i = threadIdx.x; i < n_pix_tile; i += blockDim.x) {
            float r = 0.f, g = 0.f, bl = 0.f, a = 0.f;
            uint32_t any = 0u;
            for (uint32_t k = 0; k < nk; ++k) {
                const uint32_t c = acc[bin_slot(k * n_pix_tile + i)];
                if (c) {
                    const float fc = (float)c;
                    r = __fmaf_rn(fc, prm.palette[4 * k + 0], r);
                    g = __fmaf_rn(fc, prm.palette[4 * k + 1], g);
                    bl = __fmaf_rn(fc, prm.palette[4 * k + 2], bl);
                    a = __fadd_rn(a, fc);
                    any = 1u;
                }
            }
            const uint32_t pix = (i << tshift) | tile;
            if (any && pix < n_pix) bin_red_add_v4_f32(img + 4 * (size_t)pix, r, g, bl, a);
        }
    }
}

}  // namespace cfs
