"""B200-native dark-siren hierarchical likelihood (arxiv/paper_2605_23538) -- see DESIGN.md."""
