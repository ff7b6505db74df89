"""B200-native NVFP4 GEMV hot path of arxiv/paper_2606_13233."""
