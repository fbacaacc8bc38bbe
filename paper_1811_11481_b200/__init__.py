"""B200-native per-sector TPC cellular-automaton track finder + Kalman fit (arXiv 1811.11481).

The CUDA path lives in `csrc/` behind the C-ABI of `include/tpcca.h`; `binding` is the thin
ctypes marshalling layer.  Nothing here imports `oracle/`.
"""
