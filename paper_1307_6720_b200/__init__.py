"""paper_1307_6720_b200 -- B200-native (sm_100a) multigrid solve for the poloidal potential P of
MacTaggart et al. (arXiv 1307.6720): thin Python binding over the C-ABI library `libmhs_b200.so`
(include/mhs.h).  Importing the package does not load the library; `binding` does, and fails
loudly when the CUDA extension is missing (there is no CPU fallback)."""

__all__ = ["inputs", "binding", "build"]
