// A user kernel with the luxury level baked in: rlxpp_dev::StreamT<2048> takes the 324 products of the advance from
// include/rlxpp_rows.cuh (pre-reduced rows as immediates) instead of the run-time multiplier.  The handle must have
// been created with p = 2048.  Compiled by tests/test_host_library.py; not part of the library.
#include "rlxpp_device.cuh"
#include "rlxpp_rows.cuh"

__global__ void sum_kernel(rlxpp_view_t view, double* sums, unsigned int n) {
  const unsigned long long i = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= view.n) return;
  rlxpp_dev::StreamT<2048> g;
  g.load(view, i);
  double s = 0.0;
  for (unsigned int t = 0; t < n; t++) s += g.draw();
  g.store(view, i);
  sums[i] = s;
}
