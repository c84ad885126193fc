"""B200-native (sm_100a) call-auction clearing library -- the hot path of KineticSim
(arxiv/paper_2606_21784).  See DESIGN.md.  The CUDA library is loaded lazily by `binding`;
importing the package alone needs neither a GPU nor the built library."""
__all__ = ["workloads"]
