"""pgsf-b200: B200-native hot path of the filter-based HI source finder of arXiv 1507.04941."""
