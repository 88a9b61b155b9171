// tile_pipe.cuh -- TMA-staged tile pipeline for the streaming kernels (sm_100a).
//
// Every per-call kernel of the path streams SoA rows once: for a tile of TILE consecutive events it needs the
// same TILE-element segment of R rows (cached columns, step-1 caches, decay times, weights).  One warp issues one
// bulk asynchronous copy per row segment (cp.async.bulk global -> shared, SASS UBLKCP) into one of STAGES
// shared-memory stages; the copies of a stage complete on an mbarrier (transaction count in bytes), so the loads of
// the next tiles are in flight while the block computes on the current one, with no registers or LSU slots tied up.
// Blocks are persistent: block b handles tiles b, b + gridDim.x, ...; thread tid always owns event tile*TILE + tid.
#pragma once
#include <stdint.h>

namespace tddp4k {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
// global -> shared bulk copy, completion signalled on the mbarrier; dst, src and bytes are multiples of 16
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

constexpr int PIPE_MAX_ROWS = 80;

constexpr int PIPE_MAX_ARRAYS = 6;

// What one tile consists of: n_rows row segments.  Row r is row row[r] of the SoA array arr[arr_id[r]] (row stride
// ld elements), its elements are esize[r] bytes (8: double rows, 16: double2 columns).  In a stage, row r sits at
// byte offset TILE * pre[r], pre = running sum of the element sizes.  Passed to the kernels by value.
struct RowList {
  int n_rows;
  int bytes_per_event;              // sum of esize: a stage holds TILE * bytes_per_event bytes
  const char *arr[PIPE_MAX_ARRAYS];
  uint8_t arr_id[PIPE_MAX_ROWS];
  uint8_t row[PIPE_MAX_ROWS];
  uint8_t esize[PIPE_MAX_ROWS];
  uint16_t pre[PIPE_MAX_ROWS];
  __host__ void add(int array, int r, int es) {
    arr_id[n_rows] = (uint8_t)array; row[n_rows] = (uint8_t)r; esize[n_rows] = (uint8_t)es;
    pre[n_rows] = (uint16_t)bytes_per_event;
    bytes_per_event += es;
    ++n_rows;
  }
};

template <int TILE, int STAGES>
struct TilePipe {
  uint64_t *bar;       // [STAGES] in shared memory
  char *stage;         // [STAGES][stage_bytes]
  const RowList &rows;
  int64_t n, ld;       // events, row stride (elements); ld is a multiple of 32 and >= n
  int64_t n_tiles;

  __device__ __forceinline__ TilePipe(uint64_t *bar_, char *stage_, const RowList &rows_, int64_t n_, int64_t ld_)
      : bar(bar_), stage(stage_), rows(rows_), n(n_), ld(ld_), n_tiles((n_ + TILE - 1) / TILE) {}

  // all threads of the block; ends with a block barrier
  __device__ __forceinline__ void init() {
    if (threadIdx.x == 0) {
#pragma unroll
      for (int s = 0; s < STAGES; ++s) mbar_init(bar + s, 1);
      mbar_fence_init();
    }
    __syncthreads();
  }
  // warp 0 only (all 32 lanes): start the copies of tile `tile` into stage `s`
  __device__ __forceinline__ void issue(int64_t tile, int s) {
    int64_t first = tile * TILE;
    int64_t cnt = ld - first < TILE ? ld - first : TILE;          // whole rows are readable up to ld
    int lane = threadIdx.x & 31;
    if (lane == 0) mbar_arrive_expect_tx(bar + s, (uint32_t)(cnt * rows.bytes_per_event));
    __syncwarp();
    char *dst = stage + (size_t)s * TILE * rows.bytes_per_event;
    for (int r = lane; r < rows.n_rows; r += 32) {
      int es = rows.esize[r];
      bulk_g2s(dst + TILE * (int)rows.pre[r], rows.arr[rows.arr_id[r]] + ((int64_t)rows.row[r] * ld + first) * es,
               (uint32_t)(cnt * es), bar + s);
    }
  }
  // prologue: fill the pipeline (warp 0), then every thread may start waiting
  __device__ __forceinline__ void prologue() {
    if (threadIdx.x < 32) {
#pragma unroll
      for (int s = 0; s < STAGES; ++s) {
        int64_t tile = blockIdx.x + (int64_t)s * gridDim.x;
        if (tile < n_tiles) issue(tile, s);
      }
    }
  }
  // k-th tile of this block: wait for its stage; returns the stage base
  __device__ __forceinline__ const char *wait(int64_t k) {
    int s = (int)(k % STAGES);
    mbar_wait(bar + s, (uint32_t)((k / STAGES) & 1));
    return stage + (size_t)s * TILE * rows.bytes_per_event;
  }
  // after the block barrier that ends the work on the k-th tile: refill its stage with the (k + STAGES)-th
  __device__ __forceinline__ void refill(int64_t k) {
    if (threadIdx.x < 32) {
      int64_t tile = blockIdx.x + (k + STAGES) * gridDim.x;
      if (tile < n_tiles) issue(tile, (int)(k % STAGES));
    }
  }
};

}  // namespace tddp4k
