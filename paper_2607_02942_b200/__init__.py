"""dyplan: B200-native plan enumerator for the physical-plan compiler of arxiv/paper_2607_02942."""
