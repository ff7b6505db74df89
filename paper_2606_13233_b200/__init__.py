"""B200-native NVFP4 GEMV hot path of arxiv/paper_2606_13233.

`binding` (the ctypes wrapper of include/nvfp4.h) is imported lazily so that `inputs` and
`build` stay importable before the shared library exists.
"""
