"""paper_2606_20374_b200 — B200-native hot path of ARGUS (arxiv/paper_2606_20374):
kernel-event reduction into per-(rank, step, sig) summaries + cross-rank median/MAD diagnosis.

The compute lives in csrc/ (CUDA, sm_100a) behind the C ABI of include/argus.h; `argus` is the thin
ctypes binding.  `workload` is the seeded input generator.  There is no CPU fallback."""
__version__ = "0.1.0"
