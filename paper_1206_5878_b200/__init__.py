"""B200-native orbit step of the Henon Monte Carlo method (arXiv 1206.5878).

``paper_1206_5878_b200.hmc`` is the thin binding over the C-ABI library (include/hmc.h);
``paper_1206_5878_b200.inputs`` the seeded synthetic input generator.  Importing the
package does not load CUDA; the first call into ``hmc`` does, and fails loudly if the
library is missing.
"""
__all__ = ["hmc", "inputs"]
