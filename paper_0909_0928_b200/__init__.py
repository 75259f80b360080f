"""B200-native demons deformable image registration (arxiv/paper_0909_0928).

`binding` is the ctypes front end of the C-ABI library declared in include/demons.h;
`phantoms` holds the seeded synthetic inputs (no method arithmetic); `build` compiles
libdemons.so in-tree for sm_100a.
"""
__all__ = ["binding", "phantoms", "build"]
