"""B200-native (sm_100a) sparse decode attention of Sparrow's sparse rollout (arxiv/paper_2606_08446).

``binding`` is the thin ctypes layer over libsparrow_b200.so (the product); ``workloads`` draws the seeded
synthetic inputs; ``engine`` holds buffers and chains summarize -> select -> sparse decode for a batch.
"""
__all__ = ["binding", "workloads", "engine", "build"]
