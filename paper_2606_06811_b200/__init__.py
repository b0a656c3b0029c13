"""B200-native speculative Y-drop gapped extension (arxiv/paper_2606_06811 hot path)."""
