"""paper_2606_17107_b200 -- B200-native RoPE reposition + splice for composable KV caches.

The product is the C-ABI CUDA library libkvr.so (include/kvr.h, csrc/); `kvr` is the thin ctypes
binding with the same entry-point names.  There is no CPU fallback: importing `kvr` fails loudly
if the library has not been built (python -m paper_2606_17107_b200.build, or __graft_entry__.build()).
"""
