"""B200-native Cross-Request State Packed Forward over a Unified KV Ring Buffer (ActionFlow, arxiv 2512.20276).

`inputs`  — seeded synthetic input generators (no method arithmetic; importable without CUDA).
`binding` — thin ctypes binding of include/af.h; loading it fails loudly when the CUDA library is missing.
"""
