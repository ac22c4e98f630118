"""uep — B200-native post-gating expert-load planning (after UltraEP, arxiv 2606.04101).

The product is the C-ABI library ``libuep.so`` (``include/uep.h``, sources in ``csrc/``);
``binding`` is the thin ctypes layer with the same entry-point names.  Importing the
package is cheap and needs no GPU; the first call into ``binding`` loads the shared library
and raises if it has not been built (there is NO CPU fallback).
"""
__all__ = ["binding", "synth"]
