"""B200-native coupled phase-field lattice Boltzmann step (arXiv 2003.06342): C-ABI library + binding."""
__all__ = ["workloads"]
