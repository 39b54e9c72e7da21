"""mkv — B200-native decode attention over a dynamically two-D-compressed KV cache
(MosaicKV, arxiv/paper_2607_00760): compress -> select -> PackedAttention.

    from paper_2607_00760_b200 import binding as mkv   # thin ctypes binding of libmkv.so (C ABI)
    from paper_2607_00760_b200 import synth            # seeded synthetic workloads

`binding` loads the CUDA shared library at import and raises ImportError if it has not been
built (python -m paper_2607_00760_b200.build); there is no CPU fallback.
"""
__all__ = ["binding", "synth", "build"]
