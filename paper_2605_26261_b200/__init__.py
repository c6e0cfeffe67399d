"""paper_2605_26261_b200: B200-native FTLM hot path (matrix-free Heisenberg H.v fused with
Lanczos).  The CUDA library is loaded lazily by `paper_2605_26261_b200.ftlm`; importing the
package (e.g. for `workloads`) does not touch CUDA."""
__all__ = ["workloads", "ftlm"]
