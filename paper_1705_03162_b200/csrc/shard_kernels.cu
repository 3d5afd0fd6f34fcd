// shard_kernels.cu — gather / scatter of the edge a shard hands to its neighbour between two swept phases
// (on distributed memory the swept rule exchanges once per
// phase instead of once per sub-timestep).  The edge is `count` consecutive points, starting at local point `off`
// (periodic in the shard's extended array of Next points), of every component of `nrows` rows of the inter-launch
// state; the message is one contiguous buffer [row][component][point], moved by whatever transport the caller has
// (cudaMemcpyAsync between shards of one process, NCCL send/recv between processes).
#include "internal.h"

namespace swept {
namespace {

template <class T>
__global__ void __launch_bounds__(256) shard_copy_kernel(T* r0, T* r1, T* r2, int nrows, int C, int64_t Next,
                                                         int64_t off, int count, T* buf, int pack) {
  const int64_t total = (int64_t)nrows * C * count;
  for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (int64_t)gridDim.x * blockDim.x) {
    const int j = (int)(e % count);
    const int c = (int)((e / count) % C);
    const int r = (int)(e / ((int64_t)count * C));
    T* row = r == 0 ? r0 : (r == 1 ? r1 : r2);
    int64_t x = (off + j) % Next;
    if (x < 0) x += Next;
    T* p = row + (int64_t)c * Next + x;
    if (pack) buf[e] = *p;
    else *p = buf[e];
  }
}

}  // namespace

int launch_shard_copy(const ShardCopy& a) {
  const int64_t total = (int64_t)a.nrows * a.C * a.count;
  if (total <= 0) return 0;
  const int threads = 256;
  const unsigned grid = (unsigned)((total + threads - 1) / threads < 1184 ? (total + threads - 1) / threads : 1184);
  if (a.elem == 8)
    shard_copy_kernel<unsigned long long><<<grid, threads, 0, a.stream>>>(
        (unsigned long long*)a.rows[0], (unsigned long long*)a.rows[1], (unsigned long long*)a.rows[2], a.nrows, a.C,
        a.Next, a.off, a.count, (unsigned long long*)a.buf, a.pack ? 1 : 0);
  else
    shard_copy_kernel<unsigned><<<grid, threads, 0, a.stream>>>((unsigned*)a.rows[0], (unsigned*)a.rows[1],
                                                               (unsigned*)a.rows[2], a.nrows, a.C, a.Next, a.off,
                                                               a.count, (unsigned*)a.buf, a.pack ? 1 : 0);
  return (int)cudaGetLastError();
}

}  // namespace swept
