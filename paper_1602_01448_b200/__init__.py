"""B200-native SHARP projection loop (arXiv 1602.01448): ctypes binding over the C-ABI library
`libsharp_b200.so` (include/sharp_b200.h).  The library is loaded on first use and the load fails loudly if
it has not been built (`python -c "import __graft_entry__ as g; g.build()"`); there is no CPU fallback."""
