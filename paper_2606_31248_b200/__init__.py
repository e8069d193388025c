"""B200-native StereoRoPE + 3D neighbourhood attention (STRATA hot path, arxiv/paper_2606_31248)."""
