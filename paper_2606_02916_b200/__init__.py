"""GreenGNN per-window hot-set staging, B200-native (arxiv/paper_2606_02916).

`inputs` is importable everywhere; `binding` loads the CUDA C-ABI library and fails
loudly when it has not been built (`python __graft_entry__.py build`).
"""
