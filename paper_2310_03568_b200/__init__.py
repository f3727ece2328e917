"""B200-native VJPs of scan and reduce-by-index (arxiv/paper_2310_03568).

The CUDA library is loaded lazily by :mod:`paper_2310_03568_b200.binding`; importing the
package (e.g. for :mod:`paper_2310_03568_b200.workloads`) does not need a GPU."""
