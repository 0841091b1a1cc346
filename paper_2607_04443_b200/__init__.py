"""B200-native performer hot path of Wan-Streamer v0.2 (arxiv/paper_2607_04443)."""
