"""B200-native (sm_100a) hot path of TF-regularised cone-beam CT reconstruction
(arxiv/paper_1008_2042).  The CUDA library is loaded on first use by `binding`;
importing the package (or `synthetic`) does not touch it."""

__all__ = ["synthetic", "binding"]
