"""paper_2202_13532_b200 -- B200-native (sm_100a) tensor-product DG Vlasov-Poisson hot path.

The product is the C-ABI library libdgvlasov.so (include/dgvlasov.h, csrc/); this package is the
thin ctypes/torch binding over it.  `from paper_2202_13532_b200 import api` loads the library and
fails loudly if it has not been built; there is no CPU fallback."""

__all__ = ["api", "build"]
