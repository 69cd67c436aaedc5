"""B200-native deferred hair pipeline (arxiv/paper_2607_04230)."""
