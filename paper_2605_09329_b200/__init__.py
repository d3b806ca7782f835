"""B200-native TTS online-distillation step (arxiv/paper_2605_09329).

``paper_2605_09329_b200.tts`` is the thin ctypes binding over the C-ABI library
(include/tts.h).  Importing the package does not load the CUDA library;
``tts.lib()`` does, and fails loudly if it is missing.  The seeded input recipes
live in the top-level ``workloads`` package (they serve the oracle's tests too).
"""
__all__ = ["tts", "build"]
