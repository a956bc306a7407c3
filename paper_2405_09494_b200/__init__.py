"""gwsig: B200-native GW self-energy evaluation with space-group symmetry adaptation.

``symsetup``  host pre-step (Algorithm 1, Eq. 26-27) -- numpy, no GPU needed.
``binding``   thin ctypes binding of the C-ABI library ``libgwsig.so`` (include/gwsig.h);
              importing it fails loudly when the library has not been built.
"""
__all__ = ["symsetup", "binding"]
