// A user kernel written against include/rlxpp_tile.cuh only: the Monte-Carlo estimate of pi of device_api_example.cu
// with the block-cooperative tensor-core advance (rlxpp_dev::TileStream).  A CTA is 128 threads; every thread calls
// draw() at every step, a thread that needs no number passes want = false.  Compiled by tests/test_host_library.py to
// show that the header is self-contained; not part of the library.
#include "rlxpp_tile.cuh"

__global__ void __launch_bounds__(128) pi_tile_kernel(rlxpp_view_t view, unsigned long long* hits, unsigned int tries) {
  __shared__ rlxpp_dev::TileShared sh;
  rlxpp_dev::TileStream g;
  g.begin(sh, view);
  const unsigned long long i = (unsigned long long)blockIdx.x * 128 + threadIdx.x;
  const bool live = i < view.n;
  g.load(view, i, live);
  unsigned long long h = 0;
  for (unsigned int t = 0; t < tries; t++) {
    const double x = g.draw(live), y = g.draw(live);
    h += x * x + y * y < 1.0 ? 1u : 0u;
  }
  if (live) {
    g.store(view, i);
    hits[i] = h;
  }
  g.end();
}
