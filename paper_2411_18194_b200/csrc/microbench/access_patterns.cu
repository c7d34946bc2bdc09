// access-pattern microbenchmark: how fast can CTAs shaped like the demag passes move data?
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__); return 1;}}while(0)

// generic: each CTA handles `nrow` rows of SEG float2 (SEG lanes), row r at base + r*row_stride; in-place scale.
// threads = SEG * TPR ; each thread handles rows t/SEG + TPR*u, u = 0..U-1   (nrow = TPR*U)
template <int SEG, int TPR, int U>
__global__ void __launch_bounds__(SEG*TPR) k_rows(float2* p, size_t row_stride, size_t cta_stride_x, size_t cta_stride_y, int comps, size_t comp_stride) {
  const int l = threadIdx.x % SEG, j = threadIdx.x / SEG;
  float2* b = p + blockIdx.x * cta_stride_x + blockIdx.y * cta_stride_y + l;
  for (int c = 0; c < comps; ++c) {
    float2 v[U];
#pragma unroll
    for (int u = 0; u < U; ++u) v[u] = b[c*comp_stride + (size_t)(j + TPR*u) * row_stride];
#pragma unroll
    for (int u = 0; u < U; ++u) { v[u].x = v[u].x * 1.0001f + v[(u+1)%U].y; }
#pragma unroll
    for (int u = 0; u < U; ++u) b[c*comp_stride + (size_t)(j + TPR*u) * row_stride] = v[u];
  }
}
// all comps loaded up front
template <int SEG, int TPR, int U, int C>
__global__ void __launch_bounds__(SEG*TPR) k_rows_c(float2* p, size_t row_stride, size_t cta_stride_x, size_t cta_stride_y, size_t comp_stride) {
  const int l = threadIdx.x % SEG, j = threadIdx.x / SEG;
  float2* b = p + blockIdx.x * cta_stride_x + blockIdx.y * cta_stride_y + l;
  float2 v[C][U];
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int u = 0; u < U; ++u) v[c][u] = b[c*comp_stride + (size_t)(j + TPR*u) * row_stride];
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int u = 0; u < U; ++u) { v[c][u].x = v[c][u].x * 1.0001f + v[(c+1)%C][(u+1)%U].y; }
#pragma unroll
  for (int c = 0; c < C; ++c)
#pragma unroll
    for (int u = 0; u < U; ++u) b[c*comp_stride + (size_t)(j + TPR*u) * row_stride] = v[c][u];
}

template <typename F> float timeit(F f, int it=20) {
  cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
  for (int i=0;i<3;++i) f();
  cudaEventRecord(a); for (int i=0;i<it;++i) f(); cudaEventRecord(b); cudaEventSynchronize(b);
  float ms; cudaEventElapsedTime(&ms,a,b); return ms/it;
}

int main() {
  const int xp = 272, py = 512, nz = 64, ny = 256;
  const size_t n2 = (size_t)3*nz*py*xp;  // spec2 elements
  float2* d; CK(cudaMalloc(&d, n2*sizeof(float2))); CK(cudaMemset(d, 0, n2*sizeof(float2)));
  // A: contiguous: treat as rows of 32 float2 contiguous: CTA handles 192 consecutive rows
  {
    size_t rows = n2/32; int ctas = rows/192;
    float ms = timeit([&]{ k_rows_c<32,8,8,3><<<dim3(ctas,1),256>>>(d, 32, (size_t)192*32, 0, (size_t)64*32); });
    printf("A contiguous 48KB/CTA (256thr, 24 ld/thr):      %.1f us  %.0f GB/s\n", ms*1e3, 2.0*ctas*192*32*8/ms/1e6);
  }
  // C: inner pattern: CTA (tile32 x, ky y): 3 comps x 64 rows x 256B, row stride py*xp, comp stride nz*py*xp
  {
    float ms = timeit([&]{ k_rows_c<32,8,8,3><<<dim3(8,py),256>>>(d, (size_t)py*xp, 32, xp, (size_t)nz*py*xp); });
    printf("C inner pattern 256B rows, 1.1MB stride:         %.1f us  %.0f GB/s\n", ms*1e3, 2.0*8*py*192*32*8/ms/1e6);
  }
  // C2: inner pattern with 128B rows (tile16), 256 thr = 16 seg x 16 tpr, U=4 per comp
  {
    float ms = timeit([&]{ k_rows_c<16,16,4,3><<<dim3(16,py),256>>>(d, (size_t)py*xp, 16, xp, (size_t)nz*py*xp); });
    printf("C2 inner pattern 128B rows:                      %.1f us  %.0f GB/s\n", ms*1e3, 2.0*16*py*192*16*8/ms/1e6);
  }
  // C3: inner with layout [ky][c][z][xp]: row stride xp, comp stride nz*xp, cta y stride 3*nz*xp
  {
    float ms = timeit([&]{ k_rows_c<32,8,8,3><<<dim3(8,py),256>>>(d, (size_t)xp, 32, (size_t)3*nz*xp, (size_t)nz*xp); });
    printf("C3 inner, ky-major layout (row stride 2176B):    %.1f us  %.0f GB/s\n", ms*1e3, 2.0*8*py*192*32*8/ms/1e6);
  }
  // B: mid pattern: CTA (tile16 x, slab y): 512 rows x 128B, row stride xp, slab stride py*xp; 512 thr = 16 x 32, U=16
  {
    float ms = timeit([&]{ k_rows_c<16,32,16,1><<<dim3(16,3*nz),512>>>(d, (size_t)xp, 16, (size_t)py*xp, 0); });
    printf("B mid pattern 128B rows stride 2176B (512 rows): %.1f us  %.0f GB/s\n", ms*1e3, 2.0*16*3*nz*512*16*8/ms/1e6);
  }
  // B2: mid pattern with 256B rows: 512 thr = 32 x 16, U = 32?? use U=16, two passes -> comps=2 trick: rows 0..255, 256..511
  {
    float ms = timeit([&]{ k_rows_c<32,16,16,2><<<dim3(8,3*nz),512>>>(d, (size_t)xp, 32, (size_t)py*xp, (size_t)256*xp); });
    printf("B2 mid pattern 256B rows:                        %.1f us  %.0f GB/s\n", ms*1e3, 2.0*8*3*nz*512*32*8/ms/1e6);
  }
  // B3: mid pattern on ky-major layout [ky][slab][xp]: row stride 3*nz*xp, slab stride xp
  {
    float ms = timeit([&]{ k_rows_c<16,32,16,1><<<dim3(16,3*nz),512>>>(d, (size_t)3*nz*xp, 16, (size_t)xp, 0); });
    printf("B3 mid on ky-major layout (row stride 417KB):    %.1f us  %.0f GB/s\n", ms*1e3, 2.0*16*3*nz*512*16*8/ms/1e6);
  }
  // D: tile-contiguous layout [ky][tile][slab][16]: mid CTA (tile, slab) rows of 128B at stride ntile*3nz*16, cta x stride 3nz*16, y stride 16
  {
    float ms = timeit([&]{ k_rows_c<16,32,16,1><<<dim3(16,3*nz),512>>>(d, (size_t)16*3*nz*16, (size_t)3*nz*16, 16, 0); });
    printf("D mid on tile-contiguous layout:                 %.1f us  %.0f GB/s\n", ms*1e3, 2.0*16*3*nz*512*16*8/ms/1e6);
  }

  // occupancy-limited variants: dynamic smem forces N CTAs/SM
  for (int kb : {100, 70, 50}) {
    cudaFuncSetAttribute(k_rows_c<32,8,8,3>, cudaFuncAttributeMaxDynamicSharedMemorySize, kb*1024);
    float ms = timeit([&]{ k_rows_c<32,8,8,3><<<dim3(8,py),256,kb*1024>>>(d, (size_t)py*xp, 32, xp, (size_t)nz*py*xp); });
    printf("C inner pattern, %d KB smem/CTA (256 thr):  %.1f us  %.0f GB/s\n", kb, ms*1e3, 2.0*8*py*192*32*8/ms/1e6);
  }
  for (int kb : {100, 70, 50}) {
    cudaFuncSetAttribute(k_rows_c<16,32,16,1>, cudaFuncAttributeMaxDynamicSharedMemorySize, kb*1024);
    float ms = timeit([&]{ k_rows_c<16,32,16,1><<<dim3(16,3*nz),512,kb*1024>>>(d, (size_t)xp, 16, (size_t)py*xp, 0); });
    printf("B mid pattern, %d KB smem/CTA (512 thr):    %.1f us  %.0f GB/s\n", kb, ms*1e3, 2.0*16*3*nz*512*16*8/ms/1e6);
  }
  printf("done\n");
  return 0;
}
