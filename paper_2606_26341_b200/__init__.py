"""jipm: B200-native batched interior-point NLP solver (hot path of arxiv 2606.26341).

``workloads`` is importable without the CUDA extension; ``jipm`` (the binding) loads the C-ABI library
lazily and fails loudly if it is missing -- there is no CPU fallback.
"""
