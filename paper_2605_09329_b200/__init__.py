"""B200-native TTS online-distillation step (arxiv/paper_2605_09329).

``paper_2605_09329_b200.tts`` is the thin ctypes binding over the C-ABI library
(include/tts.h); ``paper_2605_09329_b200.synth`` holds the seeded input recipes.
Importing the package does not load the CUDA library; ``tts.lib()`` does, and
fails loudly if it is missing.
"""
__all__ = ["synth", "tts", "build"]
