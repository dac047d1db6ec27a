// Diagnostic (not part of libhubbard_b200): what does the B200 memory system do for the access SHAPES the two
// gather sweeps of variant GATHER generate (kernels_gather.cuh), with no gather work at all?  One "pass" moves one
// vector of C4 in fp64 (12872^2 doubles = 1.33 GB) as 16-byte pieces, the unit the sweeps load and store.
//
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o membench_patterns paper_1204_3425_b200/diag/membench_patterns.cu
//   ./membench_patterns          (148 CTAs x 1024 threads, 4 pieces in flight per thread; median-free: 2 x 5 launches)
//
// Shapes (piece index as a function of tile and position i inside the tile, n = positions per tile):
//   0  contiguous                      tile * n + i                        a tile is one block (RT / CT layouts, reads)
//   1  transposed 32-byte sectors      (i / 2) * n_out + 2 * tile + i % 2  what the transposed stores of R = 2 do
//   2  transposed whole 128-byte lines ((i / 8) * (n_out / 2) + tile) * 8 + i % 8        (8 lanes fill a line)
//   3  32-byte sectors at a 128-byte stride inside the contiguous region of a 4-tile super-tile
//      (the read side that shape 2 would force on the other sweep)
// Results and what was concluded from them: profiles/r02_memory_patterns.md, DESIGN.md section 8.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

struct alignas(16) P { double v[2]; };

__device__ __forceinline__ int64_t addr(int shape, int64_t tile, int i, int n_in_p, int64_t n_out_p)
{
    switch (shape) {
        case 0: return tile * n_in_p + i;
        case 1: return (int64_t)(i >> 1) * n_out_p + tile * 2 + (i & 1);
        case 2: return ((int64_t)(i >> 3) * (n_out_p / 2) + tile) * 8 + (i & 7);
        default: return ((tile >> 2) * (int64_t)(n_in_p / 2) + (i >> 1)) * 8 + (tile & 3) * 2 + (i & 1);
    }
}

// up to two reads and three writes per piece; a shape < 0 switches that stream off
struct Streams { int r0, r1, w0, w1, w2, cs; };

__global__ void __launch_bounds__(1024, 1)
pattern_kernel(const P *__restrict__ a, const P *__restrict__ b, P *d0, P *d1, P *d2, int n_in_p, int64_t n_out_p, int64_t n_tiles, Streams s)
{
    double acc = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        for (int i0 = threadIdx.x; i0 < n_in_p; i0 += blockDim.x * 4) {
            P x[4], y[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = min(i0 + u * (int)blockDim.x, n_in_p - 1);
                x[u].v[0] = x[u].v[1] = y[u].v[0] = y[u].v[1] = 1.0;
                if (s.r0 >= 0) { const float4 t = __ldcs((const float4 *)(a + addr(s.r0, tile, i, n_in_p, n_out_p))); x[u] = *(const P *)&t; }
                if (s.r1 >= 0) { const float4 t = __ldcs((const float4 *)(b + addr(s.r1, tile, i, n_in_p, n_out_p))); y[u] = *(const P *)&t; }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int i = i0 + u * (int)blockDim.x;
                if (i >= n_in_p) continue;
                P r;
                r.v[0] = x[u].v[0] - 0.5 * y[u].v[0];
                r.v[1] = x[u].v[1] - 0.5 * y[u].v[1];
                acc += r.v[0] + r.v[1];
                P *dst[3] = {d0, d1, d2};
                const int ws[3] = {s.w0, s.w1, s.w2};
#pragma unroll
                for (int k = 0; k < 3; ++k)
                    if (ws[k] >= 0) {
                        P *p = dst[k] + addr(ws[k], tile, i, n_in_p, n_out_p);
                        if (s.cs) __stcs((float4 *)p, *(const float4 *)&r);
                        else *(float4 *)p = *(const float4 *)&r;
                    }
            }
        }
    }
    if (acc == 1.2345) printf("x");
}

int main()
{
    const int n = 12872;                                    // C4's 12870 rounded up to a multiple of 8
    const int64_t tiles = n / 2;
    const size_t bytes = (size_t)n * n * 8;
    P *a, *b, *c, *d;
    cudaMalloc(&a, bytes + 4096); cudaMalloc(&b, bytes + 4096); cudaMalloc(&c, bytes + 4096); cudaMalloc(&d, bytes + 4096);
    cudaMemset(a, 0, bytes); cudaMemset(b, 0, bytes);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    struct Case { Streams s; const char *name; } cases[] = {
        {{0, -1, -1, -1, -1, 1}, "read 1 contiguous"},
        {{0, 0, -1, -1, -1, 1}, "read 2 contiguous"},
        {{3, -1, -1, -1, -1, 1}, "read 1 as sectors at a 128-byte stride (super-tile)"},
        {{1, -1, -1, -1, -1, 1}, "read 1 as transposed 32-byte sectors"},
        {{-1, -1, 0, -1, -1, 1}, "write 1 contiguous"},
        {{-1, -1, 1, -1, -1, 1}, "write 1 as transposed 32-byte sectors (what the sweeps do)"},
        {{-1, -1, 1, -1, -1, 0}, "same without the evict-first hint"},
        {{-1, -1, 2, -1, -1, 1}, "write 1 as transposed whole 128-byte lines"},
        {{-1, -1, 3, -1, -1, 1}, "write 1 as sectors at a 128-byte stride (super-tile)"},
        {{-1, -1, 1, 1, -1, 1}, "write 2 as transposed 32-byte sectors"},
        {{0, 0, 0, -1, -1, 1}, "read 2 + write 1, all contiguous"},
        {{0, 0, 1, -1, -1, 1}, "read 2 contiguous + write 1 transposed sectors"},
        {{0, 0, 1, 1, -1, 1}, "read 2 contiguous + write 2 transposed sectors"},
        {{0, 0, 0, 1, 1, 1}, "ROW sweep: read q, f; write w in place, w and z transposed sectors"},
        {{0, 0, 0, 0, 0, 1}, "the same five passes, all contiguous"},
        {{0, -1, 1, -1, -1, 1}, "COL-like: read 1 contiguous + write 1 transposed sectors"},
        {{3, 3, 3, 2, 2, 1}, "ROW sweep on super-tiles: strided-sector reads, whole-line transposed writes"},
    };
    printf("one pass = %.3f GB; 148 CTAs x 1024 threads\n", bytes / 1e9);
    for (auto &cs : cases) {
        for (int rep = 0; rep < 2; ++rep) {
            cudaEventRecord(e0);
            for (int r = 0; r < 5; ++r) pattern_kernel<<<148, 1024>>>(a, b, (cs.s.r0 == 3 && cs.s.w0 == 3) ? a : c, d, c, n, n, tiles, cs.s);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
        }
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        ms /= 5;
        const int passes = (cs.s.r0 >= 0) + (cs.s.r1 >= 0) + (cs.s.w0 >= 0) + (cs.s.w1 >= 0) + (cs.s.w2 >= 0);
        printf("  %-76s %6.3f ms  %5.2f TB/s  (%d passes)\n", cs.name, ms, passes * (double)bytes / ms / 1e9, passes);
    }
    return cudaGetLastError() != cudaSuccess;
}
