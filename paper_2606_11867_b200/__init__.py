"""B200-native (sm_100a) ForeMoE micro-step plan + dispatch + combine path.

``binding`` is the thin ctypes layer over the C-ABI library ``libforemoe.so`` (include/foremoe.h);
``synth`` draws the seeded synthetic inputs; ``build`` compiles the library in-tree.
"""
__all__ = ["binding", "synth", "build"]
